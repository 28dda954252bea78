// pm_gravity.cuh -- PM-gravity particle <-> mesh kernels: Steps 1, 2 and 5 of Sec. 2 only
// (PAPER.md L95, L107), a purely additive mass deposit (L27, L51) with the cloud-in-cell kernel (R40), the
// converse mesh -> particle interpolation (L27) and the kick / drift halves of the kick-drift-kick leapfrog (L107).
// Compiled with -fmad=false: the weights, the products (w_z w_y) w_x and the sums keep the order DESIGN.md section 13
// states, so the interpolated accelerations agree with a plain sequential evaluation to the last bit.
#pragma once
#include "pm_device.cuh"

namespace pm {

// Per axis (cell-centred mesh): s = (x - x0) inv_dx - 1/2, i0 = floor(s), f = s - i0; cells i0 and i0 + 1 get 1 - f and f.
// i0 lies in [-1, n-1] for a particle inside the box: the low and high ghost layers are reached from the first and
// last half cell.
__device__ __forceinline__ void cic_axis(double x, double x0, double inv_dx, int &i0, double &w0, double &w1) {
    const double s = (x - x0) * inv_dx - 0.5;
    const double fl = floor(s);
    const double f = s - fl;
    i0 = (int)fl;
    w0 = 1.0 - f;
    w1 = f;
}

// Step 1 (Eq. 2): buffer channel `buf` (ghosted layout) += m W / V, eight fp64 REDs per particle.  One thread per
// particle: the two x-neighbours of a row are adjacent in memory (one 32-byte sector three times out of four).
__global__ void __launch_bounds__(256) k_grav_deposit(const DevP P, const double *__restrict__ px, const double *__restrict__ py,
                                                      const double *__restrict__ pz, const double *__restrict__ pm_,
                                                      long long n, const int *__restrict__ perm, double *__restrict__ buf,
                                                      int *__restrict__ err_flag) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const long long s = perm ? perm[t] : t;      // particles taken in a1 bin order (DRAM page / L2 sector locality)
    const double x = px[s], y = py[s], z = pz[s], m = pm_[s];
    int i0, j0, k0;
    double wx[2], wy[2], wz[2];
    cic_axis(x, P.x0[0], P.inv_dx, i0, wx[0], wx[1]);
    cic_axis(y, P.x0[1], P.inv_dx, j0, wy[0], wy[1]);
    cic_axis(z, P.x0[2], P.inv_dx, k0, wz[0], wz[1]);
    // the box test is the host-cell test of the exchange step (L43): floor((x - x0) inv_dx) in [0, n)
    const int ih = host_cell(x, P.x0[0], P.inv_dx), jh = host_cell(y, P.x0[1], P.inv_dx), kh = host_cell(z, P.x0[2], P.inv_dx);
    if (ih < 0 || ih >= P.nx || jh < 0 || jh >= P.ny || kh < 0 || kh >= P.nz || i0 < -1 || j0 < -1 || k0 < -1 ||
        i0 >= P.nx || j0 >= P.ny || k0 >= P.nz) {
        atomicOr(err_flag, 1);
        return;
    }
    const long long base = ghost_index(P, 0, j0, k0);
    const int ix[2] = { wrap1(i0, P.nx), wrap1(i0 + 1, P.nx) };       // x wrapped on the spot (deposit_index); y, z through the ghost layer
#pragma unroll
    for (int dk = 0; dk < 2; ++dk)
#pragma unroll
        for (int dj = 0; dj < 2; ++dj) {
            const double wzy = wz[dk] * wy[dj];
            double *row = buf + base + dk * P.pk + dj * P.pj;
#pragma unroll
            for (int di = 0; di < 2; ++di) atomicAdd(row + ix[di], m * (wzy * wx[di]) / P.V);
        }
}

// Step 5 (Eq. 6 with eta = 1, L95): rho_tot = rho_gas + folded buffer, owned cells only.  VEC = 2 uses 128-bit accesses
// (nx even; the ghosted row origin gx is even by construction).  rho_gas == nullptr: particles only.
template <int VEC>
__global__ void __launch_bounds__(256) k_grav_apply(const DevP P, const double *rho_gas, const double *__restrict__ buf,
                                                    double *rho_tot) {   // rho_gas may alias rho_tot: no __restrict__ on the two
    const long long nv = P.N / VEC;
    const int nxv = P.nx / VEC;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < nv; t += (long long)gridDim.x * blockDim.x) {
        const long long row = t / nxv;
        const int i = VEC * (int)(t - row * nxv);
        const int k = (int)(row / P.ny);
        const int j = (int)(row - (long long)k * P.ny);
        const double *b = buf + ghost_index(P, i, j, k);
        const long long q = row * P.nx + i;
        if constexpr (VEC == 2) {
            const double2 d = *reinterpret_cast<const double2 *>(b);
            double2 r = make_double2(0.0, 0.0);
            if (rho_gas) r = *reinterpret_cast<const double2 *>(rho_gas + q);
            *reinterpret_cast<double2 *>(rho_tot + q) = make_double2(r.x + d.x, r.y + d.y);
        } else {
            rho_tot[q] = (rho_gas ? rho_gas[q] : 0.0) + b[0];
        }
    }
}

// Mesh -> particle (L27) + half kick (L107): a = sum over the eight cells, k then j then i, low cell first, of
// ((w_z w_y) w_x) g_ijk at the periodically wrapped owned index; v += a dt when vx != nullptr; a stored when ax != nullptr.
__global__ void __launch_bounds__(256) k_grav_kick(const DevP P, const double *__restrict__ gx, const double *__restrict__ gy,
                                                   const double *__restrict__ gz, long long n, const double *__restrict__ px,
                                                   const double *__restrict__ py, const double *__restrict__ pz,
                                                   double *__restrict__ vx, double *__restrict__ vy, double *__restrict__ vz,
                                                   double dt, double *__restrict__ ax, double *__restrict__ ay,
                                                   double *__restrict__ az, const int *__restrict__ perm,
                                                   int *__restrict__ err_flag) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    const long long s = perm ? perm[t] : t;
    const double x = px[s], y = py[s], z = pz[s];
    int i0, j0, k0;
    double wx[2], wy[2], wz[2];
    cic_axis(x, P.x0[0], P.inv_dx, i0, wx[0], wx[1]);
    cic_axis(y, P.x0[1], P.inv_dx, j0, wy[0], wy[1]);
    cic_axis(z, P.x0[2], P.inv_dx, k0, wz[0], wz[1]);
    const int ih = host_cell(x, P.x0[0], P.inv_dx), jh = host_cell(y, P.x0[1], P.inv_dx), kh = host_cell(z, P.x0[2], P.inv_dx);
    if (ih < 0 || ih >= P.nx || jh < 0 || jh >= P.ny || kh < 0 || kh >= P.nz || i0 < -1 || j0 < -1 || k0 < -1 ||
        i0 >= P.nx || j0 >= P.ny || k0 >= P.nz) {
        atomicOr(err_flag, 1);
        return;
    }
    const int ii[2] = {wrap1(i0, P.nx), wrap1(i0 + 1, P.nx)};
    const int jj[2] = {wrap1(j0, P.ny), wrap1(j0 + 1, P.ny)};
    const int kk[2] = {wrap1(k0, P.nz), wrap1(k0 + 1, P.nz)};
    // all 24 loads first (independent addresses), then the sums in the stated order
    double fx[8], fy[8], fz[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const long long q = ((long long)kk[c >> 2] * P.ny + jj[(c >> 1) & 1]) * P.nx + ii[c & 1];
        fx[c] = __ldg(gx + q); fy[c] = __ldg(gy + q); fz[c] = __ldg(gz + q);
    }
    double a0 = 0.0, a1 = 0.0, a2 = 0.0;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const double w = (wz[c >> 2] * wy[(c >> 1) & 1]) * wx[c & 1];
        a0 = a0 + w * fx[c]; a1 = a1 + w * fy[c]; a2 = a2 + w * fz[c];
    }
    if (ax) { ax[s] = a0; ay[s] = a1; az[s] = a2; }
    if (vx) { vx[s] = vx[s] + a0 * dt; vy[s] = vy[s] + a1 * dt; vz[s] = vz[s] + a2 * dt; }
}

// Drift (L107): x += v dt, brought back into [lo, lo + n dx) by whole box lengths; a result that rounds onto the upper
// face goes to the lower face (R41).  A non-finite position is flagged (the loops below would not end on it).
__device__ __forceinline__ double drift1(double x, double v, double dt, double lo, double L, int *err_flag) {
    const double hi = lo + L;
    double xn = x + v * dt;
    if (!(fabs(xn) <= 1.79769313486231570e308)) { atomicOr(err_flag, 1); return xn; }
    if (fabs(xn - lo) > 1.0e6 * L) { atomicOr(err_flag, 1); return xn; }   // |v dt| of a million boxes: not a drift
    while (xn >= hi) xn = xn - L;
    while (xn < lo) xn = xn + L;
    return xn >= hi ? lo : xn;
}

__global__ void __launch_bounds__(256) k_drift(const DevP P, long long n, double *__restrict__ px, double *__restrict__ py,
                                               double *__restrict__ pz, const double *__restrict__ vx, const double *__restrict__ vy,
                                               const double *__restrict__ vz, double dt, int *__restrict__ err_flag) {
    const long long s = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    px[s] = drift1(px[s], vx[s], dt, P.x0[0], (double)P.nx * P.dx, err_flag);
    py[s] = drift1(py[s], vy[s], dt, P.x0[1], (double)P.ny * P.dx, err_flag);
    pz[s] = drift1(pz[s], vz[s], dt, P.x0[2], (double)P.nz * P.dx, err_flag);
}

}  // namespace pm
