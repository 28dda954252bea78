// pm_fast.cuh -- specialised deposit / return kernels for the shapes the BASELINE configs use
// (SN kernel half-width 3 with 4 sub-samples per axis; sink kernel half-width 4).  Same arithmetic contract as the
// generic kernels in pm_b200.cu (every integer decision is evaluated by the same expressions), but:
//   * box sizes are compile-time, so index decoding is multiply-shift instead of runtime division;
//   * cells are first classified, then COMPACTED with warp ballots, so the expensive work (64 sub-sample tests of a
//     boundary cell; gather / scatter of a cell with omega > 0) runs on full warps instead of diverged ones;
//   * 1/rho and 1/r are formed once per cell and multiplied (<= 1 ulp from the oracle's divisions, far inside the
//     1e-12 parity tolerance; no integer depends on them).
#pragma once
#include "pm_device.cuh"

namespace pm {

constexpr int kFastSnWarps = 8;
constexpr int kSnB = 7, kSnCells = 343, kSnNs = 4;

// Box cell (a, b, c) = (x, y, z offsets in 0..6) packed as a | b << 3 | c << 6 (< 448).
struct __align__(16) SnWarpSmem {
    double d2[3][kSnB * kSnNs];     // squared sub-sample offsets per axis
    double dmin[3][8], dmax[3][8];  // per-cell min / max of them
    double dc[3][8];                // cell-centre offsets from the particle per axis
    int off[3][8];                  // wrapped owned-index contribution per axis (x: i, y: j*nx, z: k*nx*ny)
    int goff[2][8];                 // ghosted-index contribution of y and z
    unsigned short list[352];       // boundary-cell list, then active-cell list (packed codes)
    unsigned char cnt[448];         // omega counts (0..64) by packed code
};

__device__ __forceinline__ unsigned lanemask_lt() {
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

__device__ __forceinline__ double pick3(int ax, double a, double b, double c) { return ax == 0 ? a : (ax == 1 ? b : c); }

// One warp per SN particle, particles taken in bin order (perm).
__global__ void __launch_bounds__(kFastSnWarps * 32, 3) k_deposit_sne_g3n4(const DevP P, const DevState U, const DevSNe S,
                                                                            double *__restrict__ buf, double *__restrict__ dbg,
                                                                            int *__restrict__ err, const int *__restrict__ perm) {
    __shared__ SnWarpSmem sm_all[kFastSnWarps];
    __shared__ unsigned short dec[352];          // linear box index -> packed code, shared by the CTA
    for (int c = threadIdx.x; c < kSnCells; c += blockDim.x) {
        const int a = c % 7, t = c / 7;
        dec[c] = (unsigned short)(a | ((t % 7) << 3) | ((t / 7) << 6));
    }
    __syncthreads();
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long w = (long long)blockIdx.x * kFastSnWarps + wib;
    if (w >= S.n) return;
    SnWarpSmem &sm = sm_all[wib];
    const long long s = perm[w];
    const double xs = S.x[s], ys = S.y[s], zs = S.z[s];
    const int ih = host_cell(xs, P.x0[0], P.inv_dx), jh = host_cell(ys, P.x0[1], P.inv_dx), kh = host_cell(zs, P.x0[2], P.inv_dx);
    if (ih < 0 || ih >= P.nx || jh < 0 || jh >= P.ny || kh < 0 || kh >= P.nz) {
        if (lane == 0) atomicOr(err, 1);
        return;
    }
    // ---- phase 0: per-axis tables -------------------------------------------------------------------------------
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        const int e = lane + 32 * r;
        if (e < 3 * kSnB * kSnNs) {
            const int ax = e / (kSnB * kSnNs), t = e - ax * (kSnB * kSnNs);
            const int c = t >> 2, q = t & 3;
            const double x0 = pick3(ax, P.x0[0], P.x0[1], P.x0[2]);
            const double ps = pick3(ax, xs, ys, zs);
            const int h = ax == 0 ? ih : (ax == 1 ? jh : kh);
            const double d = sub_centre(x0, h - 3 + c, q, kSnNs, P.dx) - ps;
            sm.d2[ax][t] = d * d;
        }
    }
    if (lane < 21) {
        const int ax = lane / 7, c = lane - ax * 7;
        const double x0 = pick3(ax, P.x0[0], P.x0[1], P.x0[2]);
        const double ps = pick3(ax, xs, ys, zs);
        const int h = ax == 0 ? ih : (ax == 1 ? jh : kh);
        const int n = ax == 0 ? P.nx : (ax == 1 ? P.ny : P.nz);
        const int u = h - 3 + c;                                  // unwrapped cell index
        sm.dc[ax][c] = cell_centre(x0, u, P.dx) - ps;
        const int wq = wrap1(u, n);
        sm.off[ax][c] = ax == 0 ? wq : (ax == 1 ? wq * P.nx : wq * P.nx * P.ny);
        if (ax > 0) sm.goff[ax - 1][c] = (int)((u + P.g) * (ax == 1 ? P.pj : P.pk));
    }
    __syncwarp();
    if (lane < 21) {
        const int ax = lane / 7, c = lane - ax * 7;
        const double v0 = sm.d2[ax][4 * c], v1 = sm.d2[ax][4 * c + 1], v2 = sm.d2[ax][4 * c + 2], v3 = sm.d2[ax][4 * c + 3];
        sm.dmin[ax][c] = fmin(fmin(v0, v1), fmin(v2, v3));
        sm.dmax[ax][c] = fmax(fmax(v0, v1), fmax(v2, v3));
    }
    __syncwarp();
    // ---- phase 1: classify the 343 cells; full -> 64, empty -> 0, boundary -> list ---------------------------------
    const double rk2 = P.rk2_sn;
    int nb = 0;
#pragma unroll 1
    for (int r = 0; r < 11; ++r) {
        const int c = lane + 32 * r;
        bool boundary = false;
        int pc = 0;
        if (c < kSnCells) {
            pc = dec[c];
            const int a = pc & 7, b = (pc >> 3) & 7, cc = pc >> 6;
            const bool full = (sm.dmax[2][cc] + sm.dmax[1][b]) + sm.dmax[0][a] <= rk2;
            const bool empty = (sm.dmin[2][cc] + sm.dmin[1][b]) + sm.dmin[0][a] > rk2;
            boundary = !full && !empty;
            sm.cnt[pc] = full ? 64 : 0;
        }
        const unsigned m = __ballot_sync(0xffffffffu, boundary);
        if (boundary) sm.list[nb + __popc(m & lanemask_lt())] = (unsigned short)pc;
        nb += __popc(m);
    }
    __syncwarp();
    // ---- phase 2: the 64 sub-sample tests of every boundary cell ---------------------------------------------------
#pragma unroll 1
    for (int idx = lane; idx < nb; idx += 32) {
        const int pc = sm.list[idx];
        const int a = pc & 7, b = (pc >> 3) & 7, cc = pc >> 6;
        const double x0 = sm.d2[0][4 * a], x1 = sm.d2[0][4 * a + 1], x2 = sm.d2[0][4 * a + 2], x3 = sm.d2[0][4 * a + 3];
        double yv[4], zv[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) { yv[q] = sm.d2[1][4 * b + q]; zv[q] = sm.d2[2][4 * cc + q]; }
        int cnt = 0;
#pragma unroll
        for (int qz = 0; qz < 4; ++qz)
#pragma unroll
            for (int qy = 0; qy < 4; ++qy) {
                const double sy = zv[qz] + yv[qy];
                cnt += ((sy + x0) <= rk2) + ((sy + x1) <= rk2) + ((sy + x2) <= rk2) + ((sy + x3) <= rk2);
            }
        sm.cnt[pc] = (unsigned char)cnt;
    }
    __syncwarp();
    // ---- phase 3: list of cells with omega > 0 -------------------------------------------------------------------
    int na = 0;
#pragma unroll 1
    for (int r = 0; r < 11; ++r) {
        const int c = lane + 32 * r;
        const int pc = c < kSnCells ? dec[c] : 0;
        const bool act = c < kSnCells && sm.cnt[pc] != 0;
        const unsigned m = __ballot_sync(0xffffffffu, act);
        if (act) sm.list[na + __popc(m & lanemask_lt())] = (unsigned short)pc;
        na += __popc(m);
    }
    __syncwarp();
    // ---- phase 4: stencil sums (O4) --------------------------------------------------------------------------------
    const double vsx = S.vx[s], vsy = S.vy[s], vsz = S.vz[s], e_sn = S.e_sn[s], m_ej = S.m_ej[s];
    double m_gas = 0.0, px = 0.0, py = 0.0, pz = 0.0, v_snr = 0.0;
#pragma unroll 1
    for (int idx = lane; idx < na; idx += 32) {
        const int pc = sm.list[idx];
        const int a = pc & 7, b = (pc >> 3) & 7, cc = pc >> 6;
        const double omega = (double)sm.cnt[pc] * (1.0 / 64.0);         // exact: power of two
        const int q = sm.off[2][cc] + sm.off[1][b] + sm.off[0][a];
        const double rho = U.rho[q], mx = U.mx[q], my = U.my[q], mz = U.mz[q];
        const double rinv = 1.0 / rho;
        const double mcell = omega * rho * P.V;
        m_gas += mcell;
        px += mcell * (mx * rinv);
        py += mcell * (my * rinv);
        pz += mcell * (mz * rinv);
        v_snr += omega * P.V;
    }
    m_gas = warp_sum(m_gas); px = warp_sum(px); py = warp_sum(py); pz = warp_sum(pz); v_snr = warp_sum(v_snr);
    const SnScalars sc = sn_scalars(P, m_gas, px, py, pz, v_snr, vsx, vsy, vsz, e_sn, m_ej);
    // ---- phase 5: Eq. 17 and the atomic additions (O5) -----------------------------------------------------------
    const double inv_vsnr = 1.0 / sc.v_snr;
    const double e_dens = (e_sn + sc.e_kin);
    double *const sbuf = buf + P.Nb + (ih - 3 + P.gx);
#pragma unroll 1
    for (int idx = lane; idx < na; idx += 32) {
        const int pc = sm.list[idx];
        const int a = pc & 7, b = (pc >> 3) & 7, cc = pc >> 6;
        const double omega = (double)sm.cnt[pc] * (1.0 / 64.0);
        const int q = sm.off[2][cc] + sm.off[1][b] + sm.off[0][a];
        const double rho = U.rho[q], mx = U.mx[q], my = U.my[q], mz = U.mz[q];
        const double rinv = 1.0 / rho;
        const double vx = mx * rinv, vy = my * rinv, vz = mz * rinv;
        const double ddx = sm.dc[0][a], ddy = sm.dc[1][b], ddz = sm.dc[2][cc];
        const double r2 = dist2(ddx, ddy, ddz);
        const double ir = r2 > 0.0 ? rsqrt(r2) : 0.0;                  // rhat = 0 at r = 0 (R21)
        const double drho = omega * m_ej * inv_vsnr;
        const double pscale = (sc.p_rad * inv_vsnr) * omega * ir;
        const double prx = pscale * ddx, pry = pscale * ddy, prz = pscale * ddz;
        const double wr = omega * rho;
        double *dst = sbuf + (sm.goff[1][cc] + sm.goff[0][b] + a);
        atomicAdd(dst, drho);
        atomicAdd(dst + P.Nb, wr * (sc.vcx - vx) + drho * sc.vcx + prx);
        atomicAdd(dst + 2 * P.Nb, wr * (sc.vcy - vy) + drho * sc.vcy + pry);
        atomicAdd(dst + 3 * P.Nb, wr * (sc.vcz - vz) + drho * sc.vcz + prz);
        atomicAdd(dst + 4 * P.Nb, omega * e_dens * inv_vsnr + ((sc.vcx * prx + sc.vcy * pry) + sc.vcz * prz));
    }
    if (dbg && lane == 0) {
        const long long n = S.n;
        dbg[s] = sc.m_snr; dbg[n + s] = sc.v_snr; dbg[2 * n + s] = sc.vcx; dbg[3 * n + s] = sc.vcy; dbg[4 * n + s] = sc.vcz;
        dbg[5 * n + s] = sc.n_h; dbg[6 * n + s] = sc.r_m; dbg[7 * n + s] = sc.p_rad; dbg[8 * n + s] = (double)sc.regime;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Sinks with kernel half-width 4 (9^3 box).  Pass A finds the member cells (r^2 <= r_K^2), sums the kernel means and
// compacts the members into a list; passes B and C (Gaussian normalisation, deposit) and the return pass run on it.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kFastSinkWarps = 4;
constexpr int kSkB = 9, kSkCells = 729;

struct __align__(16) SinkWarpSmem { unsigned short list[736]; };

__device__ __forceinline__ double sink_r2_g4(const DevP &P, int c, int ih, int jh, int kh, double xs, double ys, double zs,
                                             int &i, int &j, int &k) {
    const int a = c % 9, t = c / 9, b = t % 9, cc = t / 9;
    i = ih - 4 + a; j = jh - 4 + b; k = kh - 4 + cc;
    return dist2(cell_centre(P.x0[0], i, P.dx) - xs, cell_centre(P.x0[1], j, P.dx) - ys, cell_centre(P.x0[2], k, P.dx) - zs);
}

// member list of one sink; returns the member count (same on all lanes)
__device__ __forceinline__ int sink_member_list_g4(const DevP &P, SinkWarpSmem &sm, int lane, int ih, int jh, int kh,
                                                   double xs, double ys, double zs) {
    int nm = 0;
#pragma unroll 1
    for (int r = 0; r < 23; ++r) {
        const int c = lane + 32 * r;
        bool mem = false;
        if (c < kSkCells) {
            int i, j, k;
            mem = sink_r2_g4(P, c, ih, jh, kh, xs, ys, zs, i, j, k) <= P.rk2_sink;
        }
        const unsigned m = __ballot_sync(0xffffffffu, mem);
        if (mem) sm.list[nm + __popc(m & lanemask_lt())] = (unsigned short)c;
        nm += __popc(m);
    }
    __syncwarp();
    return nm;
}

__global__ void __launch_bounds__(kFastSinkWarps * 32) k_deposit_sinks_g4(const DevP P, const DevState U, const DevSinks S,
                                                                          const double dt, double *__restrict__ buf0,
                                                                          double *__restrict__ scal, double *__restrict__ dbg,
                                                                          int *__restrict__ err, const int *__restrict__ perm) {
    __shared__ SinkWarpSmem sm_all[kFastSinkWarps];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long w = (long long)blockIdx.x * kFastSinkWarps + wib;
    if (w >= S.n) return;
    SinkWarpSmem &sm = sm_all[wib];
    const long long s = perm[w];
    const double xs = S.x[s], ys = S.y[s], zs = S.z[s];
    const int ih = host_cell(xs, P.x0[0], P.inv_dx), jh = host_cell(ys, P.x0[1], P.inv_dx), kh = host_cell(zs, P.x0[2], P.inv_dx);
    if (ih < 0 || ih >= P.nx || jh < 0 || jh >= P.ny || kh < 0 || kh >= P.nz) {
        if (lane == 0) { atomicOr(err, 1); scal[s] = 0.0; scal[S.n + s] = 1.0; scal[2 * S.n + s] = 1.0; }
        return;
    }
    const double vsx = S.vx[s], vsy = S.vy[s], vsz = S.vz[s], ms = S.m[s];
    const int nm = sink_member_list_g4(P, sm, lane, ih, jh, kh, xs, ys, zs);
    double sum_rho = 0.0, srx = 0.0, sry = 0.0, srz = 0.0, src = 0.0;
#pragma unroll 1
    for (int idx = lane; idx < nm; idx += 32) {
        int i, j, k;
        sink_r2_g4(P, sm.list[idx], ih, jh, kh, xs, ys, zs, i, j, k);
        const long long q = owned_index(P, i, j, k);
        const double rho = U.rho[q];
        const double rinv = 1.0 / rho;
        const double cs = sound_speed(P, rho, U.eint[q]);
        sum_rho += rho;
        srx += rho * (U.mx[q] * rinv - vsx);
        sry += rho * (U.my[q] * rinv - vsy);
        srz += rho * (U.mz[q] * rinv - vsz);
        src += rho * cs;
    }
    sum_rho = warp_sum(sum_rho); srx = warp_sum(srx); sry = warp_sum(sry); srz = warp_sum(srz); src = warp_sum(src);
    const SinkScalars sc = sink_scalars(P, sum_rho, srx, sry, srz, src, nm, ms);
    const double ra2 = sc.r_acc * sc.r_acc;
    double wsum = 0.0;
#pragma unroll 1
    for (int idx = lane; idx < nm; idx += 32) {
        int i, j, k;
        const double r2 = sink_r2_g4(P, sm.list[idx], ih, jh, kh, xs, ys, zs, i, j, k);
        wsum += exp(-r2 / ra2);
    }
    wsum = warp_sum(wsum);
#pragma unroll 1
    for (int idx = lane; idx < nm; idx += 32) {
        int i, j, k;
        const double r2 = sink_r2_g4(P, sm.list[idx], ih, jh, kh, xs, ys, zs, i, j, k);
        atomicAdd(buf0 + ghost_index(P, i, j, k), -sink_cell_amount(P, r2, sc.r_acc, wsum, sc.mdot, dt));
    }
    if (lane == 0) {
        scal[s] = sc.mdot; scal[S.n + s] = sc.r_acc; scal[2 * S.n + s] = wsum;
        if (dbg) {
            const long long n = S.n;
            dbg[s] = sc.rho_inf; dbg[n + s] = sc.v_inf; dbg[2 * n + s] = sc.c_inf; dbg[3 * n + s] = sc.r_bh;
            dbg[4 * n + s] = sc.mdot; dbg[5 * n + s] = sc.r_acc; dbg[6 * n + s] = wsum; dbg[7 * n + s] = (double)nm;
        }
    }
}

__global__ void __launch_bounds__(kFastSinkWarps * 32) k_return_sinks_g4(const DevP P, const DevSinks S, const double dt,
                                                                         const double *__restrict__ scal,
                                                                         const double *__restrict__ ret,
                                                                         const int *__restrict__ perm) {
    __shared__ SinkWarpSmem sm_all[kFastSinkWarps];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long w = (long long)blockIdx.x * kFastSinkWarps + wib;
    if (w >= S.n) return;
    SinkWarpSmem &sm = sm_all[wib];
    const long long s = perm[w];
    const double xs = S.x[s], ys = S.y[s], zs = S.z[s];
    const int ih = host_cell(xs, P.x0[0], P.inv_dx), jh = host_cell(ys, P.x0[1], P.inv_dx), kh = host_cell(zs, P.x0[2], P.inv_dx);
    if (ih < 0 || ih >= P.nx || jh < 0 || jh >= P.ny || kh < 0 || kh >= P.nz) return;
    const double mdot = scal[s], r_acc = scal[S.n + s], wsum = scal[2 * S.n + s];
    const int nm = sink_member_list_g4(P, sm, lane, ih, jh, kh, xs, ys, zs);
    double dm = 0.0, dpx = 0.0, dpy = 0.0, dpz = 0.0;
#pragma unroll 1
    for (int idx = lane; idx < nm; idx += 32) {
        int i, j, k;
        const double r2 = sink_r2_g4(P, sm.list[idx], ih, jh, kh, xs, ys, zs, i, j, k);
        const double amt = sink_cell_amount(P, r2, r_acc, wsum, mdot, dt);
        if (amt > 0.0) {
            const long long q = owned_index(P, i, j, k);
            const double gain = ret[q] * amt * P.V;
            dm += gain;
            dpx += gain * ret[P.N + q];
            dpy += gain * ret[2 * P.N + q];
            dpz += gain * ret[3 * P.N + q];
        }
    }
    dm = warp_sum(dm); dpx = warp_sum(dpx); dpy = warp_sum(dpy); dpz = warp_sum(dpz);
    if (lane == 0) {
        const double m_old = S.m[s], m_new = m_old + dm;
        S.vx[s] = (m_old * S.vx[s] + dpx) / m_new;
        S.vy[s] = (m_old * S.vy[s] + dpy) / m_new;
        S.vz[s] = (m_old * S.vz[s] + dpz) / m_new;
        S.m[s] = m_new;
        if (S.dm) S.dm[s] = dm;
        if (S.dpx) S.dpx[s] = dpx;
        if (S.dpy) S.dpy[s] = dpy;
        if (S.dpz) S.dpz[s] = dpz;
    }
}

}  // namespace pm
