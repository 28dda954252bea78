// pm_sink_fast.cuh -- specialised sink deposit (a1-a3) and return (a8) kernels for kernel half-width 4 (9^3 box),
// the shape every BASELINE config uses.  Membership is the same bit-exact test as the generic kernels,
// (dz^2 + dy^2) + dx^2 <= r_K^2 on cell-centre offsets, but evaluated by ROW (81 rows of 9 cells, one row per lane,
// squared offsets tabulated per axis); members are compacted into a list of packed (a, b, c) codes.
// The Gaussian weight is separable, exp(-r^2/r_acc^2) = e_z e_y e_x, so a sink costs 27 exponentials instead of one
// per member cell per pass (the product differs from the oracle's single exp by a few ulp plus the same
// conditioning term r^2/r_acc^2 * eps both carry).  No division per cell:
// sum rho (v - v_s) = sum (m - rho v_s), rho c_s = sqrt(gamma (gamma - 1) e_int rho), a = w * [mdot dt / (V sum w)].
#pragma once
#include "pm_device.cuh"
#include "pm_tiles.cuh"

namespace pm {

constexpr int kFastSinkWarps = 4;
constexpr int kFastSinkMinBlocks = 10;   // 48 registers, 40 warps per SM (1 / 10 / 12 / 16 measured: 0.66 / 0.53 / 0.56 / 0.61 ms)
constexpr int kSkB = 9, kSkRows = 81, kSkMaxMembers = 512;   // members lie within r_K + sqrt(3)/2 cells: < 484

struct __align__(16) SinkWarpSmem {
    double d2[3][10];                  // squared cell-centre offsets per axis
    double ex[3][10];                  // exp(-d2 / r_acc^2) per axis
    int off[3][10];                    // wrapped owned-index contribution per axis
    int goff[2][10];                   // ghosted-index contribution of y and z
    unsigned short code[kSkMaxMembers];  // a | b << 4 | c << 8
};

// Tables, row masks, member list.  Returns the member count (same on all lanes).
__device__ __forceinline__ int sink_member_list_g4(const DevP &P, SinkWarpSmem &sm, int lane, int ih, int jh, int kh,
                                                   double xs, double ys, double zs) {
    if (lane < 27) {
        const int ax = lane / 9, c = lane - ax * 9;
        const double x0 = ax == 0 ? P.x0[0] : (ax == 1 ? P.x0[1] : P.x0[2]);
        const double ps = ax == 0 ? xs : (ax == 1 ? ys : zs);
        const int h = ax == 0 ? ih : (ax == 1 ? jh : kh);
        const int n = ax == 0 ? P.nx : (ax == 1 ? P.ny : P.nz);
        const int u = h - 4 + c;
        const double d = cell_centre(x0, u, P.dx) - ps;
        sm.d2[ax][c] = d * d;
        const int wq = (ax == 2) ? state_k(P, u) : wrap1(u, n);
        sm.off[ax][c] = ax == 0 ? wq : (ax == 1 ? wq * P.nx : wq * P.nx * P.ny);
        if (ax > 0) sm.goff[ax - 1][c] = (int)((u + P.g) * (ax == 1 ? P.pj : P.pk));
    }
    __syncwarp();
    const double rk2 = P.rk2_sink;
    unsigned mask[3];
    int mine = 0;
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        const int r = lane + 32 * t;
        unsigned m = 0;
        if (r < kSkRows) {
            const int b = r % 9, c = r / 9;
            const double sy = sm.d2[2][c] + sm.d2[1][b];
#pragma unroll
            for (int a = 0; a < 9; ++a) m |= ((sy + sm.d2[0][a]) <= rk2 ? 1u : 0u) << a;
        }
        mask[t] = m;
        mine += __popc(m);
    }
    int incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    const int nm = __shfl_sync(0xffffffffu, incl, 31);
    int pos = incl - mine;
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        const int r = lane + 32 * t;
        if (mask[t]) {
            const int b = r % 9, c = r / 9;
            const int crow = (b << 4) | (c << 8);
#pragma unroll
            for (int a = 0; a < 9; ++a)
                if (mask[t] >> a & 1) {
                    sm.code[pos] = (unsigned short)(crow | a);
                    ++pos;
                }
        }
    }
    __syncwarp();
    return nm;
}

// per-axis Gaussian factors (Eq. 9, separable)
__device__ __forceinline__ void sink_axis_weights(SinkWarpSmem &sm, int lane, double r_acc) {
    const double ra2 = r_acc * r_acc;
    if (lane < 27) {
        const int ax = lane / 9, c = lane - ax * 9;
        sm.ex[ax][c] = exp(-sm.d2[ax][c] / ra2);
    }
    __syncwarp();
}

__device__ __forceinline__ int sink_owned(const SinkWarpSmem &sm, int code) {
    return sm.off[2][code >> 8] + sm.off[1][(code >> 4) & 15] + sm.off[0][code & 15];
}
__device__ __forceinline__ int sink_ghosted(const SinkWarpSmem &sm, int code) {
    return sm.goff[1][code >> 8] + sm.goff[0][(code >> 4) & 15] + sm.off[0][code & 15];     // x wrapped into [0, nx) (deposit_index)
}

__device__ __forceinline__ double sink_weight(const SinkWarpSmem &sm, int code) {
    return (sm.ex[2][code >> 8] * sm.ex[1][(code >> 4) & 15]) * sm.ex[0][code & 15];
}

template <bool REPRO, bool TL>
__global__ void __launch_bounds__(kFastSinkWarps * 32, kFastSinkMinBlocks) k_deposit_sinks_g4(const DevP P, const DevState U, const DevSinks S,
                                                                          const double dt, double *__restrict__ buf0,
                                                                          double *__restrict__ scal, double *__restrict__ dbg,
                                                                          int *__restrict__ err, const int *__restrict__ perm,
                                                                          double *__restrict__ ret_tr) {
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
    // ---- O2: kernel means ------------------------------------------------------------------------------------------
    const double gg = P.gamma * (P.gamma - 1.0);
    double sum_rho = 0.0, srx = 0.0, sry = 0.0, srz = 0.0, src = 0.0;
#pragma unroll 2
    for (int i = lane; i < nm; i += 32) {
        const int q = sink_owned(sm, sm.code[i]);
        const double rho = U.rho[q], mx = U.mx[q], my = U.my[q], mz = U.mz[q];
        sum_rho += rho;
        srx += fma(-rho, vsx, mx);                 // rho (v - v_s) = m - rho v_s
        sry += fma(-rho, vsy, my);
        srz += fma(-rho, vsz, mz);
        if (P.cs_iso > 0.0) src = fma(rho, P.cs_iso, src);
        else src += sqrt(gg * U.eint[q] * rho);    // rho c_s with c_s^2 = gamma (gamma - 1) e_int / rho
    }
    sum_rho = warp_sum(sum_rho); srx = warp_sum(srx); sry = warp_sum(sry); srz = warp_sum(srz); src = warp_sum(src);
    const SinkScalars sc = sink_scalars(P, sum_rho, srx, sry, srz, src, nm, ms);
    // ---- O3: Gaussian weights, normalisation, deposit ------------------------------------------------------------------
    sink_axis_weights(sm, lane, sc.r_acc);
    double wsum = 0.0;
    for (int i = lane; i < nm; i += 32) wsum += sink_weight(sm, sm.code[i]);
    wsum = warp_sum(wsum);
    const double k = sc.mdot * dt / (wsum * P.V);         // a = mdot (w / sum w) dt / V
    double *const sbuf = buf0 + P.gx;
    for (int i = lane; i < nm; i += 32) {
        const int code = sm.code[i];
        double *dst = sbuf + sink_ghosted(sm, code);
        double amt = sink_weight(sm, code) * k;
        if (TL) {                                       // Eqs. 13-14: max(mdot_BH, mdot_Tr) phi dt / V = max(a, rho - rho_Tr)
            const int q = sink_owned(sm, code);
            amt = fmax(amt, truelove_excess(P, U.rho[q], U.eint[q]));
            ret_tr[q] = -CUDART_INF;                    // invalidate last step's entry; the apply pass rewrites it where mass is removed
        }
        red_add(dst, -amt);                           // R1: signed
        if (REPRO) red_add(dst + kChK * P.Nb, kSinkUnit);   // Appendix A: contribution count (same-sign terms: T = |sum|)
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

__global__ void __launch_bounds__(kFastSinkWarps * 32, kFastSinkMinBlocks) k_return_sinks_g4(const DevP P, const DevSinks S, const double dt,
                                                                         const double *__restrict__ scal,
                                                                         const double *__restrict__ ret,
                                                                         const double *__restrict__ ret_tr,
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
    sink_axis_weights(sm, lane, r_acc);
    const double kV = (mdot * dt / (wsum * P.V)) * P.V;   // gain = eta a V
    double dm = 0.0, dpx = 0.0, dpy = 0.0, dpz = 0.0;
#pragma unroll 2
    for (int i = lane; i < nm; i += 32) {
        const int code = sm.code[i];
        const int q = sink_owned(sm, code);
        double aV = sink_weight(sm, code) * kV;                              // a V
        if (ret_tr) aV = fmax(aV, ret_tr[q] * P.V);                          // Eq. 14 from the pre-step rho - rho_Tr
        if (aV > 0.0) {                         // a == 0 deposited nothing, so the return mesh has no entry there
            const double2 *r = reinterpret_cast<const double2 *>(ret + 4 * (long long)q);   // (eta, v_old): one sector
            const double2 r0 = r[0], r1 = r[1];
            const double gain = r0.x * aV;
            dm += gain;
            dpx = fma(gain, r0.y, dpx);
            dpy = fma(gain, r1.x, dpy);
            dpz = fma(gain, r1.y, dpz);
        }
    }
    dm = warp_sum(dm); dpx = warp_sum(dpx); dpy = warp_sum(dpy); dpz = warp_sum(dpz);
    if (lane == 0) {
        const double m_old = S.m[s], m_new = m_old + dm;
        if (m_new != 0.0) {                       // R43: a massless sink that gained nothing keeps its velocity (no 0/0)
            S.vx[s] = (m_old * S.vx[s] + dpx) / m_new;
            S.vy[s] = (m_old * S.vy[s] + dpy) / m_new;
            S.vz[s] = (m_old * S.vz[s] + dpz) / m_new;
        }
        S.m[s] = m_new;
        if (S.dm) S.dm[s] = dm;
        if (S.dpx) S.dpx[s] = dpx;
        if (S.dpy) S.dpy[s] = dpy;
        if (S.dpz) S.dpz[s] = dpz;
    }
}

}  // namespace pm
