// pm_tiles.cuh -- buffer reset (a0, L59 "all cells initialized to zero") by 8^3-cell tiles with liveness flags.
//
// The buffer mesh is cut into tiles of 8 x 8 x 8 cells; every tile carries one flag byte (bit 0: channel group K, bit 1: group
// N).  After the particles of a step have been binned (a1), k_tiles_mark rewrites ALL flags: a tile is LIVE in a group when some
// particle of this step can add into it -- decided from the occupancy of the 8^3 particle bins, no particle is looked at again
// -- and the reset stores zeros into the live tiles only.  A tile that is not live is STALE: it holds whatever an earlier step
// left there, and every reader (fold, apply, sink creation) takes it as zeros WITHOUT loading it.  A step that touches 6 % of the
// mesh (BASELINE config 4) resets and reads 6 % of the buffer; a step that touches all of it (config 5) pays the plain sweep.
//
// (Zeroing a tile lazily, by the first warp that adds into it, was built and measured first: 10.4 ms per step at config 5
// against 9.4 ms.  With ~4700 particles in flight the zeros written by one warp are evicted from L2 before that warp's own
// additions arrive -- a probe that stores a tile's zeros and adds into it in the same warp, back to back, still misses on 49 %
// of the RED sectors at a 5 GB footprint -- so the additions fetch the zeros back from DRAM just as they do after a sweep, and
// the zeroing then sits in the particle kernel's critical path.  DESIGN.md section 6.)
//
// Channel groups: K = the accretion channel (sinks), N = the five supernova channels (+ the two Appendix A error scales); the
// Appendix A count channel is zeroed where either group is live.
//
// Tile t of an axis holds the cells [8 (t - 1), 8 t) of owned coordinates (ghost cells have i < 0 or i >= n), so owned tiles
// are aligned with the 8^3 particle bins of a1 and tile 0 is pure ghost.
#pragma once
#include "pm_device.cuh"

namespace pm {

constexpr unsigned kLiveK = 1u, kLiveN = 2u;
struct Tiles {
    unsigned char *live;      // per tile: kLiveK | kLiveN
    int *swept;               // [2]: 1 when the last reset swept the whole of group K / N (k_zero_sweep): every tile of that group then
                              // holds zeros or this step's sums, so a reader may take all of them as live without loading the flags
};
__device__ __forceinline__ bool tiles_swept(const Tiles &T, int grp) { return __ldg(T.swept + grp) != 0; }

// fp64 atomic addition without return (REDG.E.ADD.F64), the Step 1 accumulation of Eq. 2
__device__ __forceinline__ void red_add(double *p, double v) {
    asm volatile("red.relaxed.gpu.global.add.f64 [%0], %1;" :: "l"(p), "d"(v) : "memory");
}

__device__ __forceinline__ int tile_axis(int i) { return (i + 8) >> 3; }          // i >= -8
__device__ __forceinline__ int tile_index(const DevP &P, int i, int j, int k) {
    return (tile_axis(k) * P.nty + tile_axis(j)) * P.ntx + tile_axis(i);
}

// Store zeros into the channels of `chmask` of tile t (whole warp).  Rows are 64 bytes; with nx even every pair of cells is
// 16-byte aligned (the ghosted row pitch and the x origin gx are even).
__device__ __forceinline__ void tile_zero(const DevP &P, double *__restrict__ buf, int t, unsigned chmask, int lane) {
    const int tx = t % P.ntx, r = t / P.ntx, ty = r % P.nty, tz = r / P.nty;
    const int i0 = 8 * (tx - 1);
    const int ilo = max(i0, -P.gx), ihi = min(i0 + 8, P.nx + P.gx);
    const int jlo = max(8 * (ty - 1), -P.g), jhi = min(8 * ty, P.ny + P.g);
    const int klo = max(8 * (tz - 1), -P.g), khi = min(8 * tz, P.nz + P.g);
    const int nj = jhi - jlo, nk = khi - klo;
    if (nj <= 0 || nk <= 0 || ihi <= ilo) return;
    if ((P.nx & 1) == 0) {
        const double2 z = make_double2(0.0, 0.0);
        for (int it = lane; it < nj * nk * 4; it += 32) {
            const int i = i0 + 2 * (it & 3), row = it >> 2;
            if (i < ilo || i >= ihi) continue;
            const int kk = row / nj, jj = row - kk * nj;
            const long long q = ghost_index(P, i, jlo + jj, klo + kk);
            for (unsigned m = chmask; m; m &= m - 1)
                *reinterpret_cast<double2 *>(buf + (long long)(__ffs(m) - 1) * P.Nb + q) = z;
        }
    } else {
        for (int it = lane; it < nj * nk * 8; it += 32) {
            const int i = i0 + (it & 7), row = it >> 3;
            if (i < ilo || i >= ihi) continue;
            const int kk = row / nj, jj = row - kk * nj;
            const long long q = ghost_index(P, i, jlo + jj, klo + kk);
            for (unsigned m = chmask; m; m &= m - 1) buf[(long long)(__ffs(m) - 1) * P.Nb + q] = 0.0;
        }
    }
}

// Host-cell ranges (one axis) from which a particle with kernel half-width g reaches tile t: directly, or through the fold --
// the tile's owned cells within g of a face also receive what was added to their ghost images one box length away (Eq. 3).
// Writes up to three inclusive ranges of BIN indices (host cell >> 3) into lo[] / hi[]; returns their number.
// open: the axis is not periodic inside this ctx (z of a slab): no images.
__device__ __forceinline__ int tile_host_bins(int t, int n, int g, int lo[3], int hi[3], bool open = false) {
    const int a = 8 * (t - 1), b = 8 * t - 1;              // the tile's cells
    int cnt = 0;
#pragma unroll
    for (int s = -1; s <= 1; ++s) {                         // image shift s n: cells a + s n .. b + s n
        int ca = a, cb = b;
        if (s != 0) {                                       // only owned cells have images, and an image lies in [-g, n + g)
            if (open) continue;
            const int oa = max(a, 0), ob = min(b, n - 1);
            if (oa > ob) continue;
            ca = max(oa + s * n, -g); cb = min(ob + s * n, n + g - 1);
            if (ca > cb) continue;
        }
        const int ha = max(ca - g, 0), hb = min(cb + g, n - 1);     // host cells that reach [ca, cb]
        if (ha > hb) continue;
        lo[cnt] = ha >> 3; hi[cnt] = hb >> 3;
        ++cnt;
    }
    return cnt;
}

// a0, first half: one thread per tile.  occ[key] != 0 says that particle bin `key` (bin_key of a1; sinks in [0, ntile), SNe
// in [ntile, 2 ntile)) holds a particle in this step.  A tile is live when a bin that can reach it is occupied (conservative:
// the whole bin counts, not the individual boxes).  live[0] / live[1] count the live tiles per group.
__global__ void __launch_bounds__(256) k_tiles_mark(const DevP P, const Tiles T, const unsigned char *__restrict__ occ,
                                                    const int ntiles, const bool has_k, const bool has_n, int *__restrict__ live) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    bool any[2] = { false, false };
    if (t < ntiles) {
        const int tx = t % P.ntx, r = t / P.ntx, ty = r % P.nty, tz = r / P.nty;
#pragma unroll
        for (int grp = 0; grp < 2; ++grp) {
            if (grp == 0 ? !has_k : !has_n) continue;
            const int g = grp == 0 ? P.gs : P.gn;
            int xl[3], xh[3], yl[3], yh[3], zl[3], zh[3];
            const int cx = tile_host_bins(tx, P.nx, g, xl, xh), cy = tile_host_bins(ty, P.ny, g, yl, yh),
                      cz = tile_host_bins(tz, P.nz, g, zl, zh, P.zopen != 0);
            const unsigned char *o = occ + (grp == 0 ? 0 : P.ntile);
            bool hit = false;
            for (int c = 0; c < cz && !hit; ++c)
                for (int bz = zl[c]; bz <= zh[c] && !hit; ++bz)
                    for (int b = 0; b < cy && !hit; ++b)
                        for (int by = yl[b]; by <= yh[b] && !hit; ++by)
                            for (int a = 0; a < cx && !hit; ++a)
                                for (int bx = xl[a]; bx <= xh[a]; ++bx)
                                    if (o[bin_key(P, bx << 3, by << 3, bz << 3)]) { hit = true; break; }
            any[grp] = hit;
        }
        // z slab: the owned cells within g of a z face receive what the NEIGHBOUR's particles added to its ghost planes; what
        // those are is not known here, so these tiles are live in every group the run uses
        if (P.zopen && 8 * tz > 0 && 8 * (tz - 1) < P.nz && (8 * (tz - 1) < P.g || 8 * tz > P.nz - P.g)) {
            any[0] = any[0] || P.gs > 0;
            any[1] = any[1] || P.gn > 0;
        }
        T.live[t] = (unsigned char)((any[0] ? kLiveK : 0u) | (any[1] ? kLiveN : 0u));
    }
    const unsigned mk = __ballot_sync(0xffffffffu, any[0]), mn = __ballot_sync(0xffffffffu, any[1]);
    if ((threadIdx.x & 31) == 0) {
        if (mk) atomicAdd(live, __popc(mk));
        if (mn) atomicAdd(live + 1, __popc(mn));
    }
}

// a0, second half.  Two ways of storing the zeros, chosen per channel group ON THE DEVICE from the number of tiles
// k_tiles_mark found live (both kernels are always launched; the one that has nothing to do returns at once):
//   sparse group (fewer than kDenseNum / kDenseDen of the tiles live): k_tiles_zero, one warp per live tile;
//   dense group: k_zero_sweep, a linear sweep over the group's channels at the store bandwidth of the device (tile by tile,
//   64-byte row pieces, costs 1.40 ms for the whole mesh of config 5 against 1.03 ms for the sweep).  The sweep also records
//   that it ran (Tiles::swept): fold and apply then skip the flag loads of that group.
constexpr int kDenseNum = 3, kDenseDen = 5;
__device__ __forceinline__ bool group_dense(const int *__restrict__ live, int grp, int ntiles) {
    return (long long)live[grp] * kDenseDen >= (long long)ntiles * kDenseNum;
}

__global__ void __launch_bounds__(256) k_tiles_zero(const DevP P, double *__restrict__ buf, const Tiles T, const bool repro,
                                                    const int ntiles, const int *__restrict__ live) {
    const bool dk = group_dense(live, 0, ntiles), dn = group_dense(live, 1, ntiles);
    if (dk && dn) return;
    const int lane = threadIdx.x & 31, nwarps = gridDim.x * 8;
    for (int t = blockIdx.x * 8 + (threadIdx.x >> 5); t < ntiles; t += nwarps) {
        const unsigned f = T.live[t];
        const bool lk = !dk && (f & kLiveK), ln = !dn && (f & kLiveN);
        unsigned mask = 0;
        if (lk) mask |= repro ? (1u | (1u << kChK)) : 1u;
        if (ln) mask |= repro ? (0xFEu | (1u << kChK)) : 0x3Eu;
        if (mask) tile_zero(P, buf, t, mask, lane);
    }
}

__device__ __forceinline__ void zero_range(double *__restrict__ p, long long n, long long tid, long long nthreads) {
    if (n <= 0) return;
    const long long head = (reinterpret_cast<unsigned long long>(p) & 8ull) ? 1 : 0;     // 16-byte alignment of the middle part
    double2 *q = reinterpret_cast<double2 *>(p + head);
    const long long n2 = (n - head) >> 1;
    const double2 z = make_double2(0.0, 0.0);
    for (long long i = tid; i < n2; i += nthreads) q[i] = z;
    if (tid == 0) {
        if (head) p[0] = 0.0;
        if ((n - head) & 1) p[n - 1] = 0.0;
    }
}

__global__ void __launch_bounds__(256) k_zero_sweep(const DevP P, double *__restrict__ buf, const bool repro, const int ntiles,
                                                    const int *__restrict__ live, int *__restrict__ swept) {
    const bool dk = group_dense(live, 0, ntiles), dn = group_dense(live, 1, ntiles);
    if (blockIdx.x == 0 && threadIdx.x == 0) { swept[0] = dk; swept[1] = dn; }
    if (!dk && !dn) return;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x, nth = (long long)gridDim.x * blockDim.x;
    if (dk) zero_range(buf, P.Nb, tid, nth);
    if (dn) zero_range(buf + P.Nb, (repro ? 7 : 5) * P.Nb, tid, nth);
    if (repro) zero_range(buf + (long long)kChK * P.Nb, P.Nb, tid, nth);
}

}  // namespace pm
