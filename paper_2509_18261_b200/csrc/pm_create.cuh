// pm_create.cuh -- sink particle creation (Sec. 3.1.2; readings R38, R39).
// Separate find and apply kernels, because every test must see the state as it was on entry: k_create_find marks the
// cells that create a sink (rho > rho_Tr, strict local maximum among the cells within r_K, retained accretion buffer zero)
// with a flag; k_create_compact lists them in cell order (scan of per-block counts); k_create_apply makes the particles
// and lowers the cells.  Nothing but the final count goes to the host.
#pragma once
#include "pm_device.cuh"
#include "pm_tiles.cuh"

namespace pm {

// Eq. 12 with the oracle's operation order
__device__ __forceinline__ double truelove_rho(const DevP &P, double rho, double eint) {
    const double cs = sound_speed(P, rho, eint);
    return ((P.tl_num * cs) * cs) / P.tl_den;
}

// buf0 = accretion channel of the (folded, retained) buffer mesh, or nullptr when no deposit has been made yet.
// One thread per cell for tests (i) and (iii); the few cells that pass are then handled by the whole warp, one after the
// other: the 32 lanes split the (2g+1)^3 neighbour offsets and leave at the first neighbour that is not smaller -- a lone
// lane walking its 257 neighbours would hold the other 31 idle (a third of the time of the first version).
__global__ void __launch_bounds__(256) k_create_find(const DevP P, const DevState U, const double *__restrict__ buf0, const Tiles T,
                                                     unsigned char *__restrict__ flag, int *__restrict__ block_count) {
    const long long c_raw = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const bool valid = c_raw < P.N;
    const long long c = valid ? c_raw : 0;
    const double rho = U.rho[c + P.zoff];             // zoff: ghost planes of a z slab in front of the owned cells
    const int i = (int)(c % P.nx);
    const long long row = c / P.nx;
    const int j = (int)(row % P.ny), k = (int)(row / P.ny);
    bool cand = valid && rho > truelove_rho(P, rho, U.eint[c + P.zoff]);              // (i)   above rho_Tr
    // (iii) inside another sink's kernel (L177); a tile no sink touched in the last step is stale and stands for zeros
    if (cand && buf0 && (T.live[tile_index(P, i, j, k)] & kLiveK) && buf0[ghost_index(P, i, j, k)] != 0.0) cand = false;
    unsigned todo = __ballot_sync(0xffffffffu, cand);
    bool created = false;
    const int g = P.gs, B = 2 * g + 1, nb = B * B * B;
    while (todo) {
        const int src = __ffs(todo) - 1;
        todo &= todo - 1;
        const int ci = __shfl_sync(0xffffffffu, i, src), cj = __shfl_sync(0xffffffffu, j, src), ck = __shfl_sync(0xffffffffu, k, src);
        const double crho = __shfl_sync(0xffffffffu, rho, src);
        bool is_max = true;
        for (int base = 0; base < nb; base += 32) {
            const int o = base + lane;
            bool bad = false;
            if (o < nb) {
                const int di = o % B - g, t = o / B, dj = t % B - g, dk = t / B - g;
                if ((di | dj | dk) && !(dist2((double)di * P.dx, (double)dj * P.dx, (double)dk * P.dx) > P.rk2_sink))
                    bad = !(U.rho[owned_index(P, ci + di, cj + dj, ck + dk)] < crho);   // (ii) strict local maximum (R39)
            }
            if (__any_sync(0xffffffffu, bad)) { is_max = false; break; }
        }
        if (lane == src) created = is_max;
    }
    // every cell gets its flag (no separate clearing pass); the block's count feeds the ordered compaction
    if (valid) flag[c] = created ? 1 : 0;
    const int n_warp = __popc(__ballot_sync(0xffffffffu, created));
    if (lane == 0 && n_warp) atomicAdd(block_count + blockIdx.x, n_warp);
}

// Ordered compaction: block b writes its creating cells, in cell order, behind those of all earlier blocks
// (block_start = exclusive scan of the block counts, in chunks of `chunk` with chunk offsets in `sums`).
__global__ void __launch_bounds__(256) k_create_compact(long long n_cells, const unsigned char *__restrict__ flag,
                                                        const int *__restrict__ block_start, const int *__restrict__ sums, int chunk,
                                                        int *__restrict__ list, int cap, int *__restrict__ total) {
    __shared__ int warp_n[8];
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const bool f = c < n_cells && flag[c] != 0;
    const unsigned m = __ballot_sync(0xffffffffu, f);
    if (lane == 0) warp_n[wib] = __popc(m);
    __syncthreads();
    int before = 0, in_block = 0;
    for (int w = 0; w < 8; ++w) { if (w < wib) before += warp_n[w]; in_block += warp_n[w]; }
    const int base = block_start[blockIdx.x] + sums[blockIdx.x / chunk];
    if (f) {
        const int pos = base + before + __popc(m & ((1u << lane) - 1u));
        if (pos < cap) list[pos] = (int)c;
    }
    if (blockIdx.x == gridDim.x - 1 && threadIdx.x == 0) *total = base + in_block;
}

// one thread per new sink; cells sorted by index
__global__ void __launch_bounds__(128) k_create_apply(const DevP P, const DevState U, const int *__restrict__ cells, int n,
                                                      double *__restrict__ x, double *__restrict__ y, double *__restrict__ z,
                                                      double *__restrict__ vx, double *__restrict__ vy, double *__restrict__ vz,
                                                      double *__restrict__ m) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const long long c0 = cells[s];
    const int i = (int)(c0 % P.nx);
    const long long row = c0 / P.nx;
    const int j = (int)(row % P.ny), k = (int)(row / P.ny);
    const long long c = c0 + P.zoff;
    const double rho = U.rho[c];
    const double rtr = truelove_rho(P, rho, U.eint[c]);
    const double keep = rtr / rho;                       // same velocity and specific energies (L183)
    x[s] = cell_centre(P.x0[0], i, P.dx); y[s] = cell_centre(P.x0[1], j, P.dx); z[s] = cell_centre(P.x0[2], k, P.dx);
    vx[s] = U.mx[c] / rho; vy[s] = U.my[c] / rho; vz[s] = U.mz[c] / rho;
    m[s] = (rho - rtr) * P.V;
    U.rho[c] = rtr;
    U.mx[c] *= keep; U.my[c] *= keep; U.mz[c] *= keep; U.etot[c] *= keep; U.eint[c] *= keep;
}

}  // namespace pm
