// pm_create.cuh -- sink particle creation (Sec. 3.1.2; readings R38, R39).
// Two kernels, because every test must see the state as it was on entry: k_create_find marks the cells that create a
// sink (rho > rho_Tr, strict local maximum among the cells within r_K, retained accretion buffer zero) and appends them
// to a list; the host sorts the (short) list by cell index; k_create_apply makes the particles and lowers the cells.
#pragma once
#include "pm_device.cuh"

namespace pm {

// Eq. 12 with the oracle's operation order
__device__ __forceinline__ double truelove_rho(const DevP &P, double rho, double eint) {
    const double cs = sound_speed(P, rho, eint);
    return ((P.tl_num * cs) * cs) / P.tl_den;
}

// buf0 = accretion channel of the (folded, retained) buffer mesh, or nullptr when no deposit has been made yet
__global__ void __launch_bounds__(256) k_create_find(const DevP P, const DevState U, const double *__restrict__ buf0,
                                                     int *__restrict__ list, int cap, int *__restrict__ count) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= P.N) return;
    const double rho = U.rho[c];
    if (!(rho > truelove_rho(P, rho, U.eint[c]))) return;                       // (i)   above rho_Tr
    const int i = (int)(c % P.nx);
    const long long row = c / P.nx;
    const int j = (int)(row % P.ny), k = (int)(row / P.ny);
    if (buf0 && buf0[ghost_index(P, i, j, k)] != 0.0) return;                    // (iii) inside another sink's kernel (L177)
    const int g = P.gs;
    for (int dk = -g; dk <= g; ++dk)
        for (int dj = -g; dj <= g; ++dj)
            for (int di = -g; di <= g; ++di) {
                if (!(di | dj | dk)) continue;
                if (dist2((double)di * P.dx, (double)dj * P.dx, (double)dk * P.dx) > P.rk2_sink) continue;
                if (!(U.rho[owned_index(P, i + di, j + dj, k + dk)] < rho)) return;   // (ii) strict local maximum (R39)
            }
    const int slot = atomicAdd(count, 1);
    if (slot < cap) list[slot] = (int)c;
}

// one thread per new sink; cells sorted by index
__global__ void __launch_bounds__(128) k_create_apply(const DevP P, const DevState U, const int *__restrict__ cells, int n,
                                                      double *__restrict__ x, double *__restrict__ y, double *__restrict__ z,
                                                      double *__restrict__ vx, double *__restrict__ vy, double *__restrict__ vz,
                                                      double *__restrict__ m) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const long long c = cells[s];
    const int i = (int)(c % P.nx);
    const long long row = c / P.nx;
    const int j = (int)(row % P.ny), k = (int)(row / P.ny);
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
