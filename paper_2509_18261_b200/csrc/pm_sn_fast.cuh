// pm_sn_fast.cuh -- specialised supernova deposit (a1, a4, a5) for kernel half-width 3 with 4 sub-samples per axis,
// the shape every BASELINE config uses.  Same arithmetic contract as the generic k_deposit_sne (every omega count is
// the exact number of sub-samples with (dz^2 + dy^2) + dx^2 <= r_K^2), but:
//   * box sizes are compile-time, so index decoding is multiply-shift instead of runtime division;
//   * cells are first classified, then COMPACTED with warp ballots, so the expensive work (64 sub-sample tests of a
//     boundary cell; gather / scatter of a cell with omega > 0) runs on full warps instead of diverged ones;
//   * no division per cell: P_gas = sum (omega V) m and omega rho (v_COM - v) = omega (rho v_COM - m); rhat = d * rsqrt(r^2);
//     value arithmetic uses explicit fma() (a few ulp from the oracle's forms, far inside the parity tolerances; no
//     integer depends on it).
// One fused kernel on purpose: its arithmetic phases (tables, classification, sub-sample tests) and its memory phases
// (gather, fp64 RED scatter) belong to different warps at any moment and overlap on the SM.  A split into a geometry
// kernel and a gather/scatter kernel was measured slower.
#pragma once
#include "pm_device.cuh"
#include "pm_tiles.cuh"

namespace pm {

// 4 warps per CTA, 8 CTAs per SM (64 registers, no spills): the kernel is latency-bound, and 32 resident warps measured
// 4.57 ms against 5.40 ms for 8 warps x 3 CTAs (74 registers); 36 and 40 warps need spills and are no faster.
constexpr int kFastSnWarps = 4;
constexpr int kFastSnMinBlocks = 8;
constexpr int kSnGatherBatch = 2;   // list entries per lane whose loads are in flight together (2 / 3 / 6 measured alike)
constexpr int kSnB = 7, kSnCells = 343, kSnNs = 4;

// Box cell (a, b, c) = (x, y, z offsets in 0..6) packed as a | b << 3 | c << 6 (< 448).
struct __align__(16) SnWarpSmem {
    double d2[3][kSnB * kSnNs];     // squared sub-sample offsets per axis
    double thr[kSnB * kSnNs];       // per x sub-sample: the largest s >= 0 with fl(s + dx^2) <= r_K^2 (-1: none)
    double dmin[3][8], dmax[3][8];  // per-cell min / max of them
    double dc[3][8];                // cell-centre offsets from the particle per axis
    int off[3][8];                  // wrapped owned-index contribution per axis (x: i, y: j*nx, z: k*nx*ny)
    unsigned short list[352];       // boundary-cell list, then active-cell list (packed codes)
    unsigned char cnt[448];         // omega counts (0..64) by packed code
};

// cnt += (s <= t), as one DSETP and one predicated add (the C form compiles to a select and costs a third instruction:
// 866 -> 590 warp instructions per particle in the 64-sample tests, the largest single item of the kernel)
__device__ __forceinline__ void count_le(int &cnt, const double s, const double t) {
    asm("{ .reg .pred p; setp.le.f64 p, %1, %2; @p add.s32 %0, %0, 1; }" : "+r"(cnt) : "d"(s), "d"(t));
}

__device__ __forceinline__ unsigned lanemask_lt() {
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// The largest double s >= 0 that passes the sub-sample test  fl(s + x) <= R  (x >= 0), or -1 when not even s = 0 passes.
// fl(s + x) is monotone in s, so the test is  s <= sn_threshold(x)  EXACTLY: the estimate R - x + h (h = half the gap
// above R, the rounding boundary) is walked to the boundary with the test itself, which makes the result independent
// of how good the estimate was.
__device__ __forceinline__ double sn_threshold(const double x, const double R) {
    if (!(x <= R)) return -1.0;
    const double h = 0.5 * (__longlong_as_double(__double_as_longlong(R) + 1) - R);
    const double hi = R - x, lo = (R - hi) - x;          // R - x = hi + lo exactly (R >= x >= 0)
    double t = hi + (lo + h);
    for (int it = 0; it < 64 && !((t + x) <= R); ++it) t = __longlong_as_double(__double_as_longlong(t) - 1);
    for (int it = 0; it < 64; ++it) {
        const double u = __longlong_as_double(__double_as_longlong(t) + 1);
        if (!((u + x) <= R)) break;
        t = u;
    }
    return t;
}

__device__ __forceinline__ double pick3(int ax, double a, double b, double c) { return ax == 0 ? a : (ax == 1 ? b : c); }

// Shared-memory-privatised tile accumulator (north_star): the five SN channels of the 14^3 cells a particle hosted in
// one 8^3 tile can reach (tile + 3-cell halo), 5 x 2744 doubles = 107 KB, owned by ONE CTA that processes all particles of
// the tile.  fp64 has no native shared-memory atomic add (atomicAdd(double*) on shared memory compiles to a CAS loop,
// ATOMS.CAST.SPIN.64), so the warps of the CTA take turns under one CTA-wide lock and add with plain loads and stores:
// 5 x (LDS, DADD, STS) per 32 cells.
constexpr int kAccSide = 14, kAccCells = kAccSide * kAccSide * kAccSide;
struct SnTileAcc {
    double *acc;        // [5][kAccCells] in shared memory
    int *lock;          // 0 = free
    int ox, oy, oz;     // owned coordinates of accumulator cell (0, 0, 0): tile origin - 3
};

// The whole deposit of ONE supernova by one warp (all 32 lanes must call).  s = particle index; sm = this warp's shared
// scratch.
template <bool REPRO, bool DENSE = false>
__device__ __forceinline__ void sn_deposit_one(const DevP &P, const DevState &U, const DevSNe &S, double *__restrict__ buf,
                                               double *__restrict__ dbg, int *__restrict__ err, const long long s,
                                               SnWarpSmem &sm, const int lane, const SnTileAcc *tile = nullptr) {
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
        const int wq = (ax == 2) ? state_k(P, u) : wrap1(u, n);      // z of a slab: the state holds the neighbour's planes itself
        sm.off[ax][c] = ax == 0 ? wq : (ax == 1 ? wq * P.nx : wq * P.nx * P.ny);
    }
    __syncwarp();
    if (lane < 21) {
        const int ax = lane / 7, c = lane - ax * 7;
        const double v0 = sm.d2[ax][4 * c], v1 = sm.d2[ax][4 * c + 1], v2 = sm.d2[ax][4 * c + 2], v3 = sm.d2[ax][4 * c + 3];
        sm.dmin[ax][c] = fmin(fmin(v0, v1), fmin(v2, v3));
        sm.dmax[ax][c] = fmax(fmax(v0, v1), fmax(v2, v3));
    }
    if (lane < kSnB * kSnNs) sm.thr[lane] = sn_threshold(sm.d2[0][lane], P.rk2_sn);
    __syncwarp();
    // ---- phase 1: classify by ROWS (49 rows of 7 cells; this lane owns rows `lane` and `lane + 32`): two fp64 compares per
    // cell give bit masks of the full and of the boundary cells; the boundary cells go to a list (any order)
    const double rk2 = P.rk2_sn;
    const int b0 = lane % 7, c0 = lane / 7;
    const int b1 = (lane + 32) % 7, c1 = (lane + 32) / 7;
    const bool has1 = lane < 17;
    const int code0 = (b0 << 3) | (c0 << 6), code1 = (b1 << 3) | (c1 << 6);
    unsigned fm0 = 0, bm0 = 0, fm1 = 0, bm1 = 0;
    {
        const double smax0 = sm.dmax[2][c0] + sm.dmax[1][b0], smin0 = sm.dmin[2][c0] + sm.dmin[1][b0];
        const double smax1 = has1 ? sm.dmax[2][c1] + sm.dmax[1][b1] : 0.0, smin1 = has1 ? sm.dmin[2][c1] + sm.dmin[1][b1] : 0.0;
#pragma unroll
        for (int a = 0; a < 7; ++a) {
            const double xmax = sm.dmax[0][a], xmin = sm.dmin[0][a];
            const bool f0 = (smax0 + xmax) <= rk2, e0 = (smin0 + xmin) > rk2;
            const bool f1 = (smax1 + xmax) <= rk2, e1 = (smin1 + xmin) > rk2;
            fm0 |= (f0 ? 1u : 0u) << a; bm0 |= ((!f0 && !e0) ? 1u : 0u) << a;
            fm1 |= (f1 ? 1u : 0u) << a; bm1 |= ((!f1 && !e1) ? 1u : 0u) << a;
        }
        if (!has1) { fm1 = 0; bm1 = 0; }
    }
    int nb;
    {
        const int mine = __popc(bm0) + __popc(bm1);
        int incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        nb = __shfl_sync(0xffffffffu, incl, 31);
        int pos = incl - mine;
#pragma unroll
        for (int a = 0; a < 7; ++a) if (bm0 >> a & 1) sm.list[pos++] = (unsigned short)(code0 | a);
#pragma unroll
        for (int a = 0; a < 7; ++a) if (bm1 >> a & 1) sm.list[pos++] = (unsigned short)(code1 | a);
    }
    __syncwarp();
    // ---- phase 2: the 64 sub-sample tests of every boundary cell ---------------------------------------------------
#pragma unroll 1
    for (int idx = lane; idx < nb; idx += 32) {
        const int pc = sm.list[idx];
        const int a = pc & 7, b = (pc >> 3) & 7, cc = pc >> 6;
        // (dz^2 + dy^2) + dx^2 <= r_K^2 in its exact threshold form: one add and four compares per (z, y) pair
        const double t0 = sm.thr[4 * a], t1 = sm.thr[4 * a + 1], t2 = sm.thr[4 * a + 2], t3 = sm.thr[4 * a + 3];
        double yv[4], zv[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) { yv[q] = sm.d2[1][4 * b + q]; zv[q] = sm.d2[2][4 * cc + q]; }
        int cnt = 0;
#pragma unroll
        for (int qz = 0; qz < 4; ++qz)
#pragma unroll
            for (int qy = 0; qy < 4; ++qy) {
                const double sy = zv[qz] + yv[qy];
                count_le(cnt, sy, t0); count_le(cnt, sy, t1); count_le(cnt, sy, t2); count_le(cnt, sy, t3);
            }
        sm.cnt[pc] = (unsigned char)cnt;
    }
    __syncwarp();
    // ---- phase 3: list of cells with omega > 0, whole rows kept contiguous (rows 0..31, then rows 32..48); an entry is the
    // packed code | (omega count - 1) << 9
    int na;
    {
        unsigned k0[7], k1[7];                    // omega counts of this lane's cells (0: not active)
        int n0 = 0, n1 = 0;
#pragma unroll
        for (int a = 0; a < 7; ++a) {
            k0[a] = (fm0 >> a & 1) ? 64u : ((bm0 >> a & 1) ? sm.cnt[code0 | a] : 0u);
            k1[a] = (fm1 >> a & 1) ? 64u : ((bm1 >> a & 1) ? sm.cnt[code1 | a] : 0u);
            n0 += k0[a] != 0; n1 += k1[a] != 0;
        }
        const int mine = n0 | (n1 << 16);
        int incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        const int tot = __shfl_sync(0xffffffffu, incl, 31);
        const int nA = tot & 0xffff;
        na = nA + (tot >> 16);
        int p0 = (incl - mine) & 0xffff, p1 = nA + ((incl - mine) >> 16);
        __syncwarp();                             // phase 2's reads of the boundary list are done: reuse it
#pragma unroll
        for (int a = 0; a < 7; ++a) if (k0[a]) sm.list[p0++] = (unsigned short)(code0 | a | ((k0[a] - 1) << 9));
#pragma unroll
        for (int a = 0; a < 7; ++a) if (k1[a]) sm.list[p1++] = (unsigned short)(code1 | a | ((k1[a] - 1) << 9));
    }
    __syncwarp();
    // ---- phase 4: stencil sums (O4) --------------------------------------------------------------------------------
    const double vsx = S.vx[s], vsy = S.vy[s], vsz = S.vz[s], e_sn = S.e_sn[s], m_ej = S.m_ej[s];
    const double v64 = P.V * (1.0 / 64.0);
    double m_gas = 0.0, px = 0.0, py = 0.0, pz = 0.0, v_snr = 0.0;
    // owned index of a box cell: plain strides when the box does not cross the periodic seam (warp-uniform), else the
    // wrapped per-axis tables
    const bool inner = ih >= 3 && ih + 3 < P.nx && jh >= 3 && jh + 3 < P.ny && (P.zopen || (kh >= 3 && kh + 3 < P.nz));
    const int nxny = P.nx * P.ny;
    const int qb = ((kh - 3) * P.ny + (jh - 3)) * P.nx + (ih - 3) + P.zoff;
    // batches of kSnGatherBatch list entries per lane: all their loads are in flight together (the gather is latency-bound)
#pragma unroll 1
    for (int base = lane; base < na; base += 32 * kSnGatherBatch) {
        int q[kSnGatherBatch];
        double wv[kSnGatherBatch];
#pragma unroll
        for (int u = 0; u < kSnGatherBatch; ++u) {
            const int idx = base + 32 * u;
            const bool on = idx < na;
            const int e = on ? sm.list[idx] : 0;
            const int a = e & 7, b = (e >> 3) & 7, cc = (e >> 6) & 7;
            q[u] = !on ? 0 : (inner ? qb + cc * nxny + b * P.nx + a : sm.off[2][cc] + sm.off[1][b] + sm.off[0][a]);
            wv[u] = on ? (double)((e >> 9) + 1) * v64 : 0.0;              // omega V; omega = count / 64 is exact
        }
        double rho[kSnGatherBatch], mx[kSnGatherBatch], my[kSnGatherBatch], mz[kSnGatherBatch];
#pragma unroll
        for (int u = 0; u < kSnGatherBatch; ++u) { rho[u] = U.rho[q[u]]; mx[u] = U.mx[q[u]]; my[u] = U.my[q[u]]; mz[u] = U.mz[q[u]]; }
#pragma unroll
        for (int u = 0; u < kSnGatherBatch; ++u) {
            m_gas = fma(wv[u], rho[u], m_gas);                           // P_gas = sum (omega V) m: no division by rho
            px = fma(wv[u], mx[u], px);
            py = fma(wv[u], my[u], py);
            pz = fma(wv[u], mz[u], pz);
            v_snr += wv[u];
        }
    }
    m_gas = warp_sum(m_gas); px = warp_sum(px); py = warp_sum(py); pz = warp_sum(pz); v_snr = warp_sum(v_snr);
    const SnScalars sc = sn_scalars(P, m_gas, px, py, pz, v_snr, vsx, vsy, vsz, e_sn, m_ej);
    // ---- phase 5: Eq. 17 and the atomic additions (O5) -----------------------------------------------------------
    const double inv_vsnr = 1.0 / sc.v_snr;
    const double k_rho = m_ej * inv_vsnr;                 // d rho = omega M_ej / V_snr
    const double k_e = (e_sn + sc.e_kin) * inv_vsnr;     // (E_sn + E_kin) / V_snr per unit omega
    const double k_p = sc.p_rad * inv_vsnr;
    double *const sbuf = buf + P.Nb + ((long long)(kh - 3 + P.g) * P.pk + (long long)(jh - 3 + P.g) * P.pj + (ih - 3 + P.gx));
    const int pj = (int)P.pj, pk = (int)P.pk;
    const bool xin = ih >= 3 && ih + 3 < P.nx;            // warp-uniform: the box does not cross the periodic x seam
    if (DENSE) {
        // the same values, added into the CTA's tile accumulator: all 32 lanes stay in the loop (the lock is taken per warp)
        volatile double *const acc = tile->acc;
        const int lb = ((kh - 3 - tile->oz) * kAccSide + (jh - 3 - tile->oy)) * kAccSide + (ih - 3 - tile->ox);
#pragma unroll 1
        for (int base = 0; base < na; base += 32) {
            const int idx = base + lane;
            const bool on = idx < na;
            const int e = on ? sm.list[idx] : 0;
            const int a = e & 7, b = (e >> 3) & 7, cc = (e >> 6) & 7;
            const double omega = (double)((e >> 9) + 1) * (1.0 / 64.0);
            const int q = inner ? qb + cc * nxny + b * P.nx + a : sm.off[2][cc] + sm.off[1][b] + sm.off[0][a];
            const double rho = U.rho[q], mx = U.mx[q], my = U.my[q], mz = U.mz[q];
            const double ddx = sm.dc[0][a], ddy = sm.dc[1][b], ddz = sm.dc[2][cc];
            const double r2 = dist2(ddx, ddy, ddz);
            const double ir = r2 > 0.0 ? rsqrt(r2) : 0.0;
            const double drho = omega * k_rho;
            const double pscale = (k_p * omega) * ir;
            const double prx = pscale * ddx, pry = pscale * ddy, prz = pscale * ddz;
            const double dpx = fma(omega, fma(rho, sc.vcx, -mx), fma(drho, sc.vcx, prx));
            const double dpy = fma(omega, fma(rho, sc.vcy, -my), fma(drho, sc.vcy, pry));
            const double dpz = fma(omega, fma(rho, sc.vcz, -mz), fma(drho, sc.vcz, prz));
            const double de = fma(omega, k_e, fma(sc.vcx, prx, fma(sc.vcy, pry, sc.vcz * prz)));
            const int li = lb + (cc * kAccSide + b) * kAccSide + a;
            if (lane == 0) while (atomicCAS(tile->lock, 0, 1) != 0) { }
            __syncwarp();
            if (on) {
                acc[li] += drho;
                acc[kAccCells + li] += dpx;
                acc[2 * kAccCells + li] += dpy;
                acc[3 * kAccCells + li] += dpz;
                acc[4 * kAccCells + li] += de;
            }
            __threadfence_block();
            __syncwarp();
            if (lane == 0) atomicExch(tile->lock, 0);
        }
    } else
#pragma unroll 1
    for (int idx = lane; idx < na; idx += 32) {
        const int e = sm.list[idx];
        const int a = e & 7, b = (e >> 3) & 7, cc = (e >> 6) & 7;
        const double omega = (double)((e >> 9) + 1) * (1.0 / 64.0);
        const int q = inner ? qb + cc * nxny + b * P.nx + a : sm.off[2][cc] + sm.off[1][b] + sm.off[0][a];
        const double rho = U.rho[q], mx = U.mx[q], my = U.my[q], mz = U.mz[q];
        const double ddx = sm.dc[0][a], ddy = sm.dc[1][b], ddz = sm.dc[2][cc];
        const double r2 = dist2(ddx, ddy, ddz);
        const double ir = r2 > 0.0 ? rsqrt(r2) : 0.0;                  // rhat = 0 at r = 0 (R21)
        const double drho = omega * k_rho;
        const double pscale = (k_p * omega) * ir;
        const double prx = pscale * ddx, pry = pscale * ddy, prz = pscale * ddz;
        double *dst = sbuf + (cc * pk + b * pj + (xin ? a : sm.off[0][a] - (ih - 3)));   // y, z: ghosted, plain strides; x wrapped (deposit_index)
        // omega rho (v_COM - v) = omega (rho v_COM - m): no division by rho
        const double dpx = fma(omega, fma(rho, sc.vcx, -mx), fma(drho, sc.vcx, prx));
        const double dpy = fma(omega, fma(rho, sc.vcy, -my), fma(drho, sc.vcy, pry));
        const double dpz = fma(omega, fma(rho, sc.vcz, -mz), fma(drho, sc.vcz, prz));
        const double de = fma(omega, k_e, fma(sc.vcx, prx, fma(sc.vcy, pry, sc.vcz * prz)));
        red_add(dst, drho);
        red_add(dst + P.Nb, dpx);
        red_add(dst + 2 * P.Nb, dpy);
        red_add(dst + 3 * P.Nb, dpz);
        red_add(dst + 4 * P.Nb, de);
        if (REPRO) {                                 // Appendix A: error scales and the contribution count (dst is channel 1)
            red_add(dst + (kChTp - 1) * P.Nb, (fabs(dpx) + fabs(dpy)) + fabs(dpz));
            red_add(dst + (kChTe - 1) * P.Nb, fabs(de));
            red_add(dst + (kChK - 1) * P.Nb, 1.0);
        }
    }
    if (dbg && lane == 0) {
        const long long n = S.n;
        dbg[s] = sc.m_snr; dbg[n + s] = sc.v_snr; dbg[2 * n + s] = sc.vcx; dbg[3 * n + s] = sc.vcy; dbg[4 * n + s] = sc.vcz;
        dbg[5 * n + s] = sc.n_h; dbg[6 * n + s] = sc.r_m; dbg[7 * n + s] = sc.p_rad; dbg[8 * n + s] = (double)sc.regime;
    }
}

// One warp per SN particle, particles taken in bin order (perm).
template <bool REPRO>
__global__ void __launch_bounds__(kFastSnWarps * 32, kFastSnMinBlocks) k_deposit_sne_g3n4(const DevP P, const DevState U, const DevSNe S,
                                                                            double *__restrict__ buf, double *__restrict__ dbg,
                                                                            int *__restrict__ err, const int *__restrict__ perm,
                                                                            const int *__restrict__ keys_sn, const int *__restrict__ cnt_sn,
                                                                            const int dense_min) {
    __shared__ SnWarpSmem sm_all[kFastSnWarps];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long w = (long long)blockIdx.x * kFastSnWarps + wib;
    if (w >= S.n) return;
    const int s = perm[w];
    // particles of a dense bin are left to k_deposit_sne_dense (cnt_sn == nullptr: no dense path in this launch)
    if (cnt_sn && cnt_sn[keys_sn[s] - P.ntile] >= dense_min) return;
    sn_deposit_one<REPRO>(P, U, S, buf, dbg, err, s, sm_all[wib], lane);
}

// ---------------------------------------------------------------------------------------------------------------
// Dense bins: one CTA owns an 8^3 tile with many particles, accumulates all of them in shared memory and adds the tile
// accumulator to the buffer mesh once (north_star: "a shared-memory-privatised tile accumulator for clustered particles").
// Which bins take this path is decided per bin from its particle count (kSnDenseMin): a particle costs ~183 cells x 5 = 915
// global REDs on the direct path, the flush of a tile 14^3 x 5 = 13720, break-even at 15 particles per tile in RED count;
// the accumulation under the CTA-wide lock and the lower occupancy (one CTA of 16 warps per SM) put the measured break-even
// higher.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kSnDenseWarps = 16;
#ifndef PM_SN_DENSE_MIN
#define PM_SN_DENSE_MIN 48
#endif
constexpr int kSnDenseMin = PM_SN_DENSE_MIN;

// inverse of bin_key: owned tile coordinates of an SN bin
__device__ __forceinline__ void bin_tile(const DevP &P, int key, int &tx, int &ty, int &tz) {
    const int sb = key >> (3 * kSbLog2), local = key & ((1 << (3 * kSbLog2)) - 1);
    int lx = 0, ly = 0, lz = 0;
#pragma unroll
    for (int bit = 0; bit < kSbLog2; ++bit) {
        lx |= ((local >> (3 * bit)) & 1) << bit; ly |= ((local >> (3 * bit + 1)) & 1) << bit; lz |= ((local >> (3 * bit + 2)) & 1) << bit;
    }
    const int sx = sb % P.nsbx, r = sb / P.nsbx, sy = r % P.nsby, sz = r / P.nsby;
    tx = (sx << kSbLog2) + lx; ty = (sy << kSbLog2) + ly; tz = (sz << kSbLog2) + lz;
}

// SN bins with at least kSnDenseMin particles, the fullest first (they bound the tail of the dense kernel): bins with >= 4 x
// the minimum are listed from the front, the others from the back of dense_list[0 .. ntile).
__global__ void __launch_bounds__(256) k_sn_dense_bins(const int ntile, const int *__restrict__ cnt_sn, int *__restrict__ dense_list,
                                                       int *__restrict__ dense_n) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= ntile) return;
    const int c = cnt_sn[b];
    if (c < kSnDenseMin) return;
    if (c >= 4 * kSnDenseMin) dense_list[atomicAdd(dense_n, 1)] = b;
    else dense_list[ntile - 1 - atomicAdd(dense_n + 1, 1)] = b;
}

__global__ void __launch_bounds__(kSnDenseWarps * 32, 1) k_deposit_sne_dense(const DevP P, const DevState U, const DevSNe S,
                                                                             double *__restrict__ buf, double *__restrict__ dbg,
                                                                             int *__restrict__ err, const int *__restrict__ perm,
                                                                             const int *__restrict__ start_local, const int *__restrict__ sums,
                                                                             const int *__restrict__ cnt_sn, const int *__restrict__ dense_list,
                                                                             const int *__restrict__ dense_n, int *__restrict__ next,
                                                                             const int scan_chunk, const int nk) {
    extern __shared__ __align__(16) unsigned char dsm[];
    double *acc = reinterpret_cast<double *>(dsm);
    SnWarpSmem *sm_all = reinterpret_cast<SnWarpSmem *>(dsm + (size_t)5 * kAccCells * sizeof(double));
    __shared__ int lock, item;
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int e = threadIdx.x; e < 5 * kAccCells; e += blockDim.x) acc[e] = 0.0;
    if (threadIdx.x == 0) lock = 0;
    const int n_front = dense_n[0], n_back = dense_n[1];
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) item = atomicAdd(next, 1);
        __syncthreads();
        const int it = item;
        if (it >= n_front + n_back) break;
        const int b = it < n_front ? dense_list[it] : dense_list[P.ntile - 1 - (it - n_front)];
        const int key = P.ntile + b;                                          // SN keys follow the sink keys
        const int first = start_local[key] + sums[key / scan_chunk] - nk;    // position in the SN part of perm
        const int count = cnt_sn[b];
        int tx, ty, tz;
        bin_tile(P, b, tx, ty, tz);
        SnTileAcc tile = { acc, &lock, 8 * tx - 3, 8 * ty - 3, 8 * tz - 3 };
        for (int p = wib; p < count; p += kSnDenseWarps)
            sn_deposit_one<false, true>(P, U, S, buf, dbg, err, perm[first + p], sm_all[wib], lane, &tile);
        __syncthreads();
        // flush: one RED per non-zero accumulator word, then the word is cleared for the next tile
        for (int e = threadIdx.x; e < kAccCells; e += blockDim.x) {
            const int lx = e % kAccSide, r = e / kAccSide, ly = r % kAccSide, lz = r / kAccSide;
            const int i = tile.ox + lx, j = tile.oy + ly, k = tile.oz + lz;
            if (i >= P.nx + P.g || j >= P.ny + P.g || k >= P.nz + P.g) continue;      // beyond the ghost zone (ragged last tile): never touched
            double *dst = buf + P.Nb + deposit_index(P, i, j, k);
#pragma unroll
            for (int f = 0; f < 5; ++f) {
                const double v = acc[f * kAccCells + e];
                if (v != 0.0) { red_add(dst + (long long)f * P.Nb, v); acc[f * kAccCells + e] = 0.0; }
            }
        }
    }
}

}  // namespace pm
