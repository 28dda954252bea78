// pm_device.cuh -- device-side arithmetic of the particle-mesh-particle step (sm_100a).
//
// Everything that decides an integer (host cell, stencil membership, omega sub-sample counts) is written so that
// no FMA contraction can change it: this translation unit is compiled with -fmad=false, and every expression
// below keeps the operation order stated in DESIGN.md ("Arithmetic contract").
// Citations: "L" = /root/reference/PAPER.md line, "R" = DESIGN.md reading.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include <math_constants.h>

namespace pm {

constexpr int kBufChannels = 6;      // 0: accretion d rho (signed, R1/R29); 1..5: SN d rho, d p (3), d E
constexpr int kRetWords = 4;         // eta, v_old (3)
// Appendix A mode (PM_FLAG_REPRODUCIBLE) adds three channels behind the six: two error scales and the contribution counts
constexpr int kChTp = 6;             // sum_s (|dp_x| + |dp_y| + |dp_z|) of the SN terms
constexpr int kChTe = 7;             // sum_s |dE| of the SN terms
constexpr int kChK = 8;              // contribution counts in one word: SNe + 2^20 * sinks (exact in a double; < 2^20 SNe per cell)
constexpr double kSinkUnit = 1048576.0;
constexpr int kReproChannels = 9;
constexpr int kSbLog2 = 2;           // a super-block is (2^kSbLog2)^3 tiles of 8^3 cells (1..6 measured: no difference)
constexpr double kFourPi = 12.566370614359172953850573533118;

struct DevP {
    int nx, ny, nz;
    int g;            // ghost width of the buffer mesh = max(gs, gn)
    int gx;           // x offset of the owned origin inside a ghosted row: g rounded up to even (16-byte alignment)
    int gs, gn;       // kernel half-widths in cells: ceil(r_K / dx) (L59: ghosts must contain r_K)
    int nsub, regime;
    long long pj, pk; // ghosted pitches (elements): j-stride = nx + 2gx, k-stride = (nx+2gx)(ny+2g)
    long long N, Nb;  // owned / ghosted cell counts
    double dx, inv_dx, V, x0[3];
    double G, gamma, cs_iso;
    double rk_sink, rk2_sink, rk_sn, rk2_sn;
    double lambda, fmax, rho_floor;
    double tl_num, tl_den;   // Eq. 12: rho_Tr = ((tl_num c_s) c_s) / tl_den, tl_num = (J J) pi, tl_den = (G dx) dx -- the oracle's
                             // operation order, so rho - rho_Tr is bit-identical; tl_num = 0: Truelove terms off
    double eps_k, rm_ej, rm_mc, msf_c, msf_e, psnr_c, psnr_e, mu_h, nh_unit, theta;
    double nsub3;
    int nsbx, nsby, nsbz;   // super-blocks (4x4x4 tiles of 8^3 cells) per axis: the bins particles are ordered by
    int ntile;              // bin keys per particle kind: super-blocks x tiles per super-block
    int ntx, nty, ntz;      // buffer-mesh tiles of 8^3 cells per axis, ghost tiles included (pm_tiles.cuh): tile t holds the
                            // cells [8 (t - 1), 8 t) of owned coordinates
    // z-slab decomposition (pm_slab.cuh): zopen = 1 means this ctx holds one slab of a domain cut along z.  The
    // caller's state arrays and the return mesh then carry g ghost planes below and above the nz owned ones (filled by halo
    // exchanges), so a stencil that leaves the slab in z reads the neighbour's cells in place instead of wrapping; the buffer
    // mesh's z ghost planes travel to the neighbours (Eq. 3 as the paper states it, L67-71) instead of being folded in place.
    int zopen;
    int zoff;               // cells of the state arrays before owned cell (0,0,0): g ny nx when zopen, else 0
};

struct DevState { double *rho, *mx, *my, *mz, *etot, *eint; };
struct DevSinks { long long n; const double *x, *y, *z; double *vx, *vy, *vz, *m, *dm, *dpx, *dpy, *dpz; };
struct DevSNe { long long n; const double *x, *y, *z, *vx, *vy, *vz, *e_sn, *m_ej; };

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ int warp_sum_int(int v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// Host cell {ijk}_s (L43): floor((x - x0) * inv_dx)
__device__ __forceinline__ int host_cell(double x, double x0, double inv_dx) { return (int)floor((x - x0) * inv_dx); }

// Centre of unwrapped cell i, and of sub-sample q of it (R17)
__device__ __forceinline__ double cell_centre(double x0, int i, double dx) { return x0 + ((double)i + 0.5) * dx; }
__device__ __forceinline__ double sub_centre(double x0, int i, int q, int nsub, double dx) {
    return x0 + ((double)i + ((double)q + 0.5) / (double)nsub) * dx;
}
// r^2 summed in the order z, y, x
__device__ __forceinline__ double dist2(double ddx, double ddy, double ddz) { return (ddz * ddz + ddy * ddy) + ddx * ddx; }

// periodic wrap of an index known to lie in [-n, 2n)
__device__ __forceinline__ int wrap1(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

// index into a STATE array (or the return mesh) of unwrapped cell (i, j, k): periodic wrap, except along z of a slab, where
// the array holds the neighbours' planes k in [-g, 0) and [nz, nz + g) itself
__device__ __forceinline__ int state_k(const DevP &P, int k) { return P.zopen ? k + P.g : wrap1(k, P.nz); }
__device__ __forceinline__ long long owned_index(const DevP &P, int i, int j, int k) {
    return ((long long)state_k(P, k) * P.ny + wrap1(j, P.ny)) * P.nx + wrap1(i, P.nx);
}
// ghosted index of UNWRAPPED cell (i,j,k), each in [-g, n+g)
__device__ __forceinline__ long long ghost_index(const DevP &P, int i, int j, int k) {
    return (long long)(k + P.g) * P.pk + (long long)(j + P.g) * P.pj + (i + P.gx);
}
// Where a particle ADDS: x is wrapped into [0, nx) on the spot (the mesh is periodic in x inside every ctx, also on a z slab), so
// the x ghost columns of the buffer mesh never receive anything and the fold has no x images to gather (its x faces were 32-byte
// strips at a 4 KB stride: a third of its bytes and more than half of its time).  y and z keep their ghost zones (Eq. 3).
__device__ __forceinline__ long long deposit_index(const DevP &P, int i, int j, int k) {
    return ghost_index(P, wrap1(i, P.nx), j, k);
}

// Bin key of a host cell: super-blocks in raster order, the 4x4x4 tiles inside one in Morton order.  Particles are
// processed bin by bin (a counting sort by this key, filled by atomic append -- no global comparison sort), so that
// the buffer and state sectors a particle touches are still in L2 from its neighbours.
__device__ __forceinline__ int bin_key(const DevP &P, int ih, int jh, int kh) {
    const int tx = ih >> 3, ty = jh >> 3, tz = kh >> 3;
    const int sb = ((tz >> kSbLog2) * P.nsby + (ty >> kSbLog2)) * P.nsbx + (tx >> kSbLog2);
    const int m = (1 << kSbLog2) - 1;
    const int lx = tx & m, ly = ty & m, lz = tz & m;
    int local = 0;
#pragma unroll
    for (int bit = 0; bit < kSbLog2; ++bit)
        local |= (((lx >> bit) & 1) << (3 * bit)) | (((ly >> bit) & 1) << (3 * bit + 1)) | (((lz >> bit) & 1) << (3 * bit + 2));
    return (sb << (3 * kSbLog2)) + local;
}

__device__ __forceinline__ double sound_speed(const DevP &P, double rho, double eint) {
    if (P.cs_iso > 0.0) return P.cs_iso;
    return sqrt(P.gamma * (P.gamma - 1.0) * eint / rho);
}

// ---------------------------------------------------------------------------------------------------------------
// Sink accretion (Sec. 3.1.1)
// ---------------------------------------------------------------------------------------------------------------
struct SinkScalars { double rho_inf, v_inf, c_inf, r_bh, mdot, r_acc; };

// Eq. 7, Eq. 8 (second form), Eq. 10 from the kernel sums (R4-R7)
__device__ __forceinline__ SinkScalars sink_scalars(const DevP &P, double sum_rho, double srx, double sry, double srz,
                                                    double sum_rc, int cnt, double ms) {
    SinkScalars s;
    s.rho_inf = sum_rho / (double)cnt;
    s.v_inf = sqrt((srx * srx + sry * sry) + srz * srz) / sum_rho;
    s.c_inf = sum_rc / sum_rho;
    s.r_bh = P.G * ms / (s.v_inf * s.v_inf + s.c_inf * s.c_inf);
    s.mdot = kFourPi * s.rho_inf * (s.r_bh * s.r_bh) * sqrt(P.lambda * P.lambda * (s.c_inf * s.c_inf) + s.v_inf * s.v_inf);
    if (s.r_bh < 0.25 * P.dx) s.r_acc = 0.25 * P.dx;
    else if (s.r_bh > 0.5 * P.rk_sink) s.r_acc = 0.5 * P.rk_sink;
    else s.r_acc = s.r_bh;
    return s;
}

// Eq. 12: rho - rho_Tr of a cell, the amount per unit volume the Truelove condition asks to remove (Eq. 14 times
// phi dt / V); -inf when the terms are off.
__device__ __forceinline__ double truelove_excess(const DevP &P, double rho, double eint) {
    if (!(P.tl_num > 0.0)) return -CUDART_INF;
    const double cs = sound_speed(P, rho, eint);
    return rho - ((P.tl_num * cs) * cs) / P.tl_den;
}

// Eq. 9, Eq. 11, Eq. 13 mass row (per unit volume); callers take max(this, truelove_excess) when Truelove is on
__device__ __forceinline__ double sink_cell_amount(const DevP &P, double r2, double r_acc, double wsum, double mdot, double dt) {
    double w = exp(-r2 / (r_acc * r_acc));
    double phi = w / wsum;
    return mdot * phi * dt / P.V;
}

// ---------------------------------------------------------------------------------------------------------------
// Supernova stencil weights (R17): per-warp shared tables of squared sub-sample offsets per axis
// ---------------------------------------------------------------------------------------------------------------
struct SnTables {
    double *d2[3];     // [B * nsub] squared offset of each sub-sample centre from the particle, per axis
    double *dmin[3];   // [B] min over the cell's sub-samples
    double *dmax[3];   // [B] max over the cell's sub-samples
    unsigned short *cnt;   // [B^3] omega counts
};

__host__ __device__ inline size_t sn_table_bytes(int B, int nsub) {
    size_t doubles = (size_t)3 * B * nsub + (size_t)6 * B;
    size_t bytes = doubles * 8 + (size_t)B * B * B * 2;
    return (bytes + 15) & ~(size_t)15;
}

__device__ __forceinline__ SnTables sn_tables_at(unsigned char *base, int B, int nsub) {
    SnTables t;
    double *d = reinterpret_cast<double *>(base);
    for (int a = 0; a < 3; ++a) { t.d2[a] = d; d += B * nsub; }
    for (int a = 0; a < 3; ++a) { t.dmin[a] = d; d += B; }
    for (int a = 0; a < 3; ++a) { t.dmax[a] = d; d += B; }
    t.cnt = reinterpret_cast<unsigned short *>(d);
    return t;
}

// Fill the per-axis tables (whole warp cooperates), then __syncwarp.
__device__ __forceinline__ void sn_fill_tables(const DevP &P, const SnTables &t, int lane, double xs, double ys, double zs,
                                               int ih, int jh, int kh) {
    const int B = 2 * P.gn + 1, ns = P.nsub;
    const double ps[3] = { xs, ys, zs };
    const int h[3] = { ih, jh, kh };
    for (int e = lane; e < 3 * B * ns; e += 32) {
        int ax = e / (B * ns), r = e - ax * (B * ns);
        int c = r / ns, q = r - c * ns;
        double d = sub_centre(P.x0[ax], h[ax] - P.gn + c, q, ns, P.dx) - ps[ax];
        t.d2[ax][r] = d * d;
    }
    __syncwarp();
    for (int e = lane; e < 3 * B; e += 32) {
        int ax = e / B, c = e - ax * B;
        double lo = t.d2[ax][c * ns], hi = lo;
        for (int q = 1; q < ns; ++q) { double v = t.d2[ax][c * ns + q]; lo = fmin(lo, v); hi = fmax(hi, v); }
        t.dmin[ax][c] = lo;
        t.dmax[ax][c] = hi;
    }
    __syncwarp();
}

// omega count of box cell (a,b,c) = (x,y,z offsets in [0,B)).  Exactly the number of sub-samples with
// (dz^2 + dy^2) + dx^2 <= r_K^2: the two shortcuts are exact because fp addition is monotone in each argument.
__device__ __forceinline__ int sn_omega_count(const DevP &P, const SnTables &t, int a, int b, int c) {
    const int ns = P.nsub;
    const double rk2 = P.rk2_sn;
    if ((t.dmax[2][c] + t.dmax[1][b]) + t.dmax[0][a] <= rk2) return ns * ns * ns;
    if ((t.dmin[2][c] + t.dmin[1][b]) + t.dmin[0][a] > rk2) return 0;
    int cnt = 0;
    for (int qz = 0; qz < ns; ++qz) {
        const double z2 = t.d2[2][c * ns + qz];
        for (int qy = 0; qy < ns; ++qy) {
            const double s = z2 + t.d2[1][b * ns + qy];
            for (int qx = 0; qx < ns; ++qx) cnt += ((s + t.d2[0][a * ns + qx]) <= rk2) ? 1 : 0;
        }
    }
    return cnt;
}

struct SnScalars { double m_snr, v_snr, vcx, vcy, vcz, e_kin, n_h, r_m, p_rad; int regime; };

// Eq. 18, n_H, R_M, Eqs. 19-20 from the stencil sums (R18-R20, R23-R24, R27)
__device__ __forceinline__ SnScalars sn_scalars(const DevP &P, double m_gas, double px, double py, double pz, double v_snr,
                                                double vsx, double vsy, double vsz, double e_sn, double m_ej) {
    SnScalars s;
    s.m_snr = m_gas + m_ej;
    s.v_snr = v_snr;
    s.vcx = (px + m_ej * vsx) / s.m_snr;
    s.vcy = (py + m_ej * vsy) / s.m_snr;
    s.vcz = (pz + m_ej * vsz) / s.m_snr;
    s.e_kin = 0.5 * m_ej * ((vsx * vsx + vsy * vsy) + vsz * vsz);
    s.n_h = s.m_snr / (P.mu_h * s.v_snr);
    // x^e as exp(e ln x): about 2.5x fewer instructions than pow(), a few ulp from it (|e ln x| < 2 here); x = n_H > 0
    const double ln_nh = log(s.n_h / P.nh_unit);
    double m_sf = P.msf_c * exp(P.msf_e * ln_nh);
    s.r_m = s.m_snr / m_sf;
    int regime = P.regime;
    if (regime == 0) regime = (s.r_m > P.rm_mc) ? 3 : ((s.r_m > P.rm_ej) ? 2 : 1);
    s.regime = regime;
    if (regime == 3) s.p_rad = P.psnr_c * exp(P.psnr_e * ln_nh);
    else if (regime == 2) s.p_rad = sqrt(2.0 * s.m_snr * P.eps_k * e_sn);
    else s.p_rad = 0.0;
    return s;
}

// Eq. 17 for one cell with omega > 0 (R21, R22): out = (d rho, d p, d E)
__device__ __forceinline__ void sn_cell_deposit(const DevP &P, const SnScalars &s, double xs, double ys, double zs,
                                                double e_sn, double m_ej, int i, int j, int k, int cnt,
                                                double rho, double vx, double vy, double vz, double out[5]) {
    const double omega = (double)cnt / P.nsub3;
    const double ddx = cell_centre(P.x0[0], i, P.dx) - xs;
    const double ddy = cell_centre(P.x0[1], j, P.dx) - ys;
    const double ddz = cell_centre(P.x0[2], k, P.dx) - zs;
    const double r = sqrt(dist2(ddx, ddy, ddz));
    double rhx = 0.0, rhy = 0.0, rhz = 0.0;
    if (r > 0.0) { rhx = ddx / r; rhy = ddy / r; rhz = ddz / r; }
    const double drho = omega * m_ej / s.v_snr;
    const double pscale = (s.p_rad / s.v_snr) * omega;
    const double prx = pscale * rhx, pry = pscale * rhy, prz = pscale * rhz;
    out[0] = drho;
    out[1] = omega * rho * (s.vcx - vx) + drho * s.vcx + prx;
    out[2] = omega * rho * (s.vcy - vy) + drho * s.vcy + pry;
    out[3] = omega * rho * (s.vcz - vz) + drho * s.vcz + prz;
    out[4] = omega * (e_sn + s.e_kin) / s.v_snr + ((s.vcx * prx + s.vcy * pry) + s.vcz * prz);
}

// ---------------------------------------------------------------------------------------------------------------
// Steps 3 + 5 for one cell.  u = (rho, mx, my, mz, etot, eint) in/out; b = the six buffer channels (dU^sum).
// Returns eta; *lam receives the Eq. 21 factor; *vold the pre-step velocity (only meaningful when b[0] != 0).
// ---------------------------------------------------------------------------------------------------------------
template <bool TL>
__device__ __forceinline__ double apply_cell(const DevP &P, double u[6], const double b[6], double *lam_out, double vold[3]) {
    const double a = -b[0];
    double eta = 1.0;                                   // R12
    if (a > 0.0) {                                      // Eqs. 15-16 with rho_Tr = inf (R10), generalised (R11)
        double alim = a;
        const double cap = P.fmax * u[0];
        if (cap < alim) alim = cap;
        if (TL) {                                              // compiled out when the Truelove terms are off
            const double need = truelove_excess(P, u[0], u[5]);   // Eq. 16: never leave the cell above rho_Tr ...
            if (need > alim) alim = need;
            if (alim > a) alim = a;                                //          ... but never remove more than was requested
        }
        double room = u[0] - P.rho_floor;
        if (room < 0.0) room = 0.0;
        if (room < alim) alim = room;
        eta = alim / a;
        const double rho = u[0];
        vold[0] = u[1] / rho; vold[1] = u[2] / rho; vold[2] = u[3] / rho;
        // accretion group is rank one in the cell's own state (R29): dU_f = b0 * (U_f / rho)
        const double A1 = b[0] * vold[0], A2 = b[0] * vold[1], A3 = b[0] * vold[2];
        const double A4 = b[0] * (u[4] / rho), A5 = b[0] * (u[5] / rho);
        u[0] = u[0] + eta * b[0];
        u[1] = u[1] + eta * A1;
        u[2] = u[2] + eta * A2;
        u[3] = u[3] + eta * A3;
        u[4] = u[4] + eta * A4;
        u[5] = u[5] + eta * A5;
    }
    double lam = 1.0;
    const bool touched = (b[1] != 0.0) || (b[5] != 0.0) || (b[2] != 0.0) || (b[3] != 0.0) || (b[4] != 0.0);
    if (touched) {                                      // Eq. 21 (R25), then Eq. 6 for the SN group
        const double rho1 = u[0], eint1 = u[5];
        const double rho2 = rho1 + b[1];
        const double e2 = u[4] + b[5];
        const double emin = P.theta * rho2 * (eint1 / rho1);
        const double K = 2.0 * rho2 * (e2 - emin);
        const double p1x = u[1], p1y = u[2], p1z = u[3];
        const double qx = p1x + b[2], qy = p1y + b[3], qz = p1z + b[4];
        const double q2 = (qx * qx + qy * qy) + qz * qz;
        if (!(q2 <= K)) {
            const double aa = (b[2] * b[2] + b[3] * b[3]) + b[4] * b[4];
            const double bb = (p1x * b[2] + p1y * b[3]) + p1z * b[4];
            const double cc = ((p1x * p1x + p1y * p1y) + p1z * p1z) - K;
            if (aa > 0.0) {
                const double disc = bb * bb - aa * cc;
                if (disc < 0.0) lam = 0.0;
                else {
                    lam = (-bb + sqrt(disc)) / aa;
                    if (lam < 0.0) lam = 0.0;
                    if (lam > 1.0) lam = 1.0;
                }
            }
        }
        u[0] = rho2;
        u[1] = p1x + lam * b[2];
        u[2] = p1y + lam * b[3];
        u[3] = p1z + lam * b[4];
        u[4] = e2;
        const double ke = ((u[1] * u[1] + u[2] * u[2]) + u[3] * u[3]) / (2.0 * rho2);
        double ei = e2 - ke;                            // L241
        if (ei < 0.0) ei = 0.0;
        u[5] = ei;
    }
    *lam_out = lam;
    return eta;
}

// ---------------------------------------------------------------------------------------------------------------
// Appendix A (L586-615, R34): clear the N_bit least significant mantissa bits of a buffer value x that is the sum of k
// terms with sum of magnitudes T:  N_bit = ilogb((k - 1) T) - ilogb(|x|) + 1 + M, clamped to [0, 52]  (integer arithmetic
// on binary exponents: the order-independent bound E <= eps (k - 1) T for the paper's running error sum E).
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ double repro_round(double x, double T, double k, int M) {
    if (!(k > 1.0) || x == 0.0 || !(T > 0.0)) return x;
    int nb = ilogb((k - 1.0) * T) - ilogb(fabs(x)) + 1 + M;
    if (nb <= 0) return x;
    if (nb > 52) nb = 52;
    const unsigned long long u = (unsigned long long)__double_as_longlong(x) & ~((1ull << nb) - 1ull);
    return __longlong_as_double((long long)u);
}

// split the packed count word: k_sn = low part, k_sink = multiples of 2^20
__device__ __forceinline__ void repro_counts(double k, double &ksn, double &ksk) {
    ksk = floor(k * (1.0 / kSinkUnit));
    ksn = k - ksk * kSinkUnit;
}

}  // namespace pm
