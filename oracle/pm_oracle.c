/*
 * pm_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded fp64 CPU statement of one particle-mesh-particle exchange step
 * of arxiv 2509.18261, written from the paper's definitions:
 *   Step 1  particle -> buffer mesh        Eq. 2
 *   Step 2  buffer sum                     Eq. 3  (L67-71)   -- here: periodic index wrapping, no ghosts
 *   Step 3  limiter, eta = dU_lim/dU_sum   Eq. 4  (L73-77)
 *   Step 4  limited changes -> particles   Eq. 5  (L79-87)
 *   Step 5  limited changes -> mesh        Eq. 6  (L89-93)
 * with the sink-accretion recipe of Sec. 3.1.1 (Eqs. 7-11, 13, 15-16; L115-171) and the supernova
 * recipe of Sec. 3.2.1 (Eqs. 17-21; L197-241).  Readings of silent / garbled passages are the R-numbers
 * of DESIGN.md ("Readings of the paper").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call this.
 * It shares no code, header, table or helper with the CUDA path.  No blocking, fusion or reordering:
 * particles are processed in index order, cells in (k, j, i) order, sums are plain left-to-right.
 *
 * Appendix A rounding (orc_repro_*): pinned by the permutation brute force and the worked 2-term case in tests.
 *
 * Parity unpinned (defined by DESIGN.md readings only, no independent pin exists):
 *   - rho_inf away from uniform gas (R4: arithmetic mean over member cells);
 *   - the Eq. 21 fall-back branch (R25: no admissible root => lambda = 0, e_int clipped at 0).
 *
 * Build: gcc -O2 -ffp-contract=off -fPIC -shared -o liboracle_pm.so pm_oracle.c -lm
 *
 * The "#pragma omp" lines are inert in that build (no -fopenmp: gcc skips them, the program is the sequential one above and
 * is the parity reference).  bench.py's all-host-cores timing leg ("all host cores via OpenMP
 * (omp atomic deposits, parallel cell loops)") compiles this same file a second time with -fopenmp into
 * liboracle_pm_omp.so; there the particle loops of Steps 1 and 4 and the cell loop of Steps 3 + 5 run on all cores, mesh
 * additions are "omp atomic", and sums depend on the order of the additions like the GPU's.  That build is timed, never
 * compared against.
 */
#ifndef _GNU_SOURCE
#define _GNU_SOURCE
#endif
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t nx, ny, nz;
    int32_t sn_nsub;              /* omega sub-samples per axis (R17) */
    int32_t sn_regime;            /* 0 auto, 1 EJ, 2 ST, 3 MC */
    int32_t pad_;
    double dx;
    double x0[3];
    double G, gamma, cs_iso;      /* cs_iso > 0: constant sound speed (R6) */
    double rk_sink, rk_sn;        /* kernel radii r_K in length units (L117, L201) */
    double bondi_lambda;          /* lambda = e^{3/2}/4 (L130) */
    double f_max_remove;          /* max removable mass fraction per step (L161: 0.25; R11) */
    double rho_floor;             /* density floor (BASELINE.json) */
    double sn_eps_k, sn_rm_ej, sn_rm_mc;                 /* 0.28, 0.027, 1 (L223-225) */
    double sn_msf_coeff, sn_msf_exp;                     /* M_sf = coeff * (n_H/unit)^exp (L203) */
    double sn_psnr_coeff, sn_psnr_exp;                   /* Eq. 20 */
    double sn_mu_h, sn_nh_unit;
    double sn_eint_theta;         /* R25: e_min = theta * rho_2 * (e_int,1 / rho_1) */
    double truelove_J;            /* Jeans number J of Eq. 12 (0.25 in the paper, L148); 0 = Truelove terms off (R10) */
} orc_params;

/* gas state, nx*ny*nz each, x fastest, no ghosts */
typedef struct { double *rho, *mx, *my, *mz, *etot, *eint; } orc_state;

typedef struct {
    int64_t n;
    double *x, *y, *z, *vx, *vy, *vz, *m;
    /* optional per-sink diagnostics (may be NULL) */
    double *rho_inf, *v_inf, *c_inf, *r_bh, *mdot, *r_acc, *wsum;
    double *dm, *dpx, *dpy, *dpz;          /* amounts actually returned to the particle (Eq. 5) */
    int32_t *n_member;
    double *dpabs;                         /* error scale only (may be NULL): sum over the member cells of gain * (|vx| + |vy| + |vz|) */
} orc_sinks;

typedef struct {
    int64_t n;
    double *x, *y, *z, *vx, *vy, *vz, *e_sn, *m_ej;
    /* optional per-SN diagnostics (may be NULL) */
    double *m_snr, *v_snr, *vcx, *vcy, *vcz, *n_h, *r_m, *p_rad;
    int32_t *regime;                       /* 1 EJ, 2 ST, 3 MC */
} orc_sne;

/* optional cell-wise outputs of one step (any pointer may be NULL) */
typedef struct {
    double *A[6];        /* signed accretion changes dU^sum (rho, mx, my, mz, etot, eint), <= 0 for rho (R1) */
    double *S[5];        /* SN changes dU^sum (rho, mx, my, mz, etot) */
    double *Aabs[6];     /* sum over particles of |terms added| per channel (Appendix A error scale, L610; R36) */
    double *Sabs[5];
    double *eta;         /* Eq. 4 ratio for the accretion group */
    double *lam;         /* Eq. 21 lambda for the SN momentum (1 where no SN touches) */
    int32_t *sn_count;   /* number of SN particles contributing to the cell */
    int32_t *sink_count; /* number of sinks contributing to the cell */
    double *Tp;          /* Appendix A (L600-606): sum over SNe of |dp_x^s| + |dp_y^s| + |dp_z^s|, the magnitudes of the values ADDED */
    double *Te;          /* ... and of |dE^s|; one addition per particle and cell, as in the paper's E update */
    double *Scond[5];    /* error scale only (L610, R36): how strongly the cell's SN terms depend on the ROUNDING of v_COM, which is a
                          * cancelling stencil sum (Eq. 18): sum_s (omega rho + d rho) * [sum_cells omega rho V |v|]_s / M_snr,s for the
                          * momentum channels, sum_s |p_rad| . (the same) for d E; [0] unused.  May be NULL. */
} orc_mesh_out;

#define FOUR_PI 12.566370614359172953850573533118

static inline int64_t wrap(int64_t i, int64_t n) { int64_t r = i % n; return r < 0 ? r + n : r; }

static inline int64_t cell_index(const orc_params *p, int64_t i, int64_t j, int64_t k) {
    return (wrap(k, p->nz) * (int64_t)p->ny + wrap(j, p->ny)) * (int64_t)p->nx + wrap(i, p->nx);
}

/* O1 host cell (L43): i_s = floor((x_s - x0) * inv_dx), inv_dx = 1/dx computed once */
static inline int64_t host_cell(double x, double x0, double inv_dx) { return (int64_t)floor((x - x0) * inv_dx); }

static inline int kernel_halfwidth(double rk, double dx) { return (int)ceil(rk / dx); }

/* centre of (unwrapped) cell i along one axis */
static inline double cell_centre(double x0, int64_t i, double dx) { return x0 + ((double)i + 0.5) * dx; }

/* centre of sub-sample q (0..nsub-1) of (unwrapped) cell i along one axis (R17) */
static inline double sub_centre(double x0, int64_t i, int q, int nsub, double dx) {
    return x0 + ((double)i + ((double)q + 0.5) / (double)nsub) * dx;
}

/* squared distance, summed in the loop-nest order z, y, x */
static inline double dist2(double ddx, double ddy, double ddz) { return (ddz * ddz + ddy * ddy) + ddx * ddx; }

/* sound speed of a cell (R6): c_s^2 = gamma (gamma-1) e_int / rho, or the constant cs_iso */
static inline double sound_speed(const orc_params *p, double rho, double eint) {
    if (p->cs_iso > 0.0) return p->cs_iso;
    return sqrt(p->gamma * (p->gamma - 1.0) * eint / rho);
}

/* ------------------------------------------------------------------------------------------ */
/* Sink accretion, Sec. 3.1.1                                                                   */
/* ------------------------------------------------------------------------------------------ */
typedef struct {
    int64_t ih, jh, kh;       /* host cell (unwrapped == wrapped, particle inside the box) */
    int g;
    int32_t n_member;
    double rho_inf, v_inf, c_inf, r_bh, mdot, r_acc, wsum;
} sink_scalars;

/* Membership (L51-53, R2): cell centre within r_K, inclusive, tested as r^2 <= r_K^2. */
static inline int sink_member(const orc_params *p, double xs, double ys, double zs,
                              int64_t i, int64_t j, int64_t k, double *r2_out) {
    double ddx = cell_centre(p->x0[0], i, p->dx) - xs;
    double ddy = cell_centre(p->x0[1], j, p->dx) - ys;
    double ddz = cell_centre(p->x0[2], k, p->dx) - zs;
    double r2 = dist2(ddx, ddy, ddz);
    *r2_out = r2;
    return r2 <= p->rk_sink * p->rk_sink;
}

/* O2: kernel means (L121; R4-R7), Eq. 7, Eq. 8 (second form), Eq. 10; Eq. 9/11 normalisation. */
static void sink_compute_scalars(const orc_params *p, const orc_state *U, double xs, double ys, double zs,
                                 double vsx, double vsy, double vsz, double ms, sink_scalars *o) {
    const double inv_dx = 1.0 / p->dx;
    o->ih = host_cell(xs, p->x0[0], inv_dx);
    o->jh = host_cell(ys, p->x0[1], inv_dx);
    o->kh = host_cell(zs, p->x0[2], inv_dx);
    o->g = kernel_halfwidth(p->rk_sink, p->dx);
    const int g = o->g;
    double sum_rho = 0.0, sum_rvx = 0.0, sum_rvy = 0.0, sum_rvz = 0.0, sum_rc = 0.0;
    int32_t cnt = 0;
    for (int64_t k = o->kh - g; k <= o->kh + g; ++k)
        for (int64_t j = o->jh - g; j <= o->jh + g; ++j)
            for (int64_t i = o->ih - g; i <= o->ih + g; ++i) {
                double r2;
                if (!sink_member(p, xs, ys, zs, i, j, k, &r2)) continue;
                int64_t c = cell_index(p, i, j, k);
                double rho = U->rho[c];
                double vx = U->mx[c] / rho, vy = U->my[c] / rho, vz = U->mz[c] / rho;
                double cs = sound_speed(p, rho, U->eint[c]);
                sum_rho += rho;
                sum_rvx += rho * (vx - vsx);
                sum_rvy += rho * (vy - vsy);
                sum_rvz += rho * (vz - vsz);
                sum_rc += rho * cs;
                cnt += 1;
            }
    o->n_member = cnt;
    o->rho_inf = sum_rho / (double)cnt;                                          /* R4 */
    o->v_inf = sqrt((sum_rvx * sum_rvx + sum_rvy * sum_rvy) + sum_rvz * sum_rvz) / sum_rho;   /* R5 */
    o->c_inf = sum_rc / sum_rho;                                                 /* R6 */
    o->r_bh = p->G * ms / (o->v_inf * o->v_inf + o->c_inf * o->c_inf);           /* Eq. 7 */
    o->mdot = FOUR_PI * o->rho_inf * (o->r_bh * o->r_bh) *
              sqrt(p->bondi_lambda * p->bondi_lambda * (o->c_inf * o->c_inf) + o->v_inf * o->v_inf);  /* Eq. 8 */
    /* Eq. 10 */
    if (o->r_bh < 0.25 * p->dx) o->r_acc = 0.25 * p->dx;
    else if (o->r_bh > 0.5 * p->rk_sink) o->r_acc = 0.5 * p->rk_sink;
    else o->r_acc = o->r_bh;
    /* Eq. 9 summed over the kernel (denominator of Eq. 11) */
    double wsum = 0.0;
    for (int64_t k = o->kh - g; k <= o->kh + g; ++k)
        for (int64_t j = o->jh - g; j <= o->jh + g; ++j)
            for (int64_t i = o->ih - g; i <= o->ih + g; ++i) {
                double r2;
                if (!sink_member(p, xs, ys, zs, i, j, k, &r2)) continue;
                wsum += exp(-r2 / (o->r_acc * o->r_acc));
            }
    o->wsum = wsum;
}

/* Eq. 12: rho_Tr = J^2 pi c_s^2 / (G dx^2) with the cell's own sound speed (R6); +inf when the terms are off (R10). */
static inline double rho_truelove(const orc_params *p, double rho, double eint) {
    if (!(p->truelove_J > 0.0)) return INFINITY;
    double cs = sound_speed(p, rho, eint);
    return p->truelove_J * p->truelove_J * M_PI * cs * cs / (p->G * p->dx * p->dx);
}

/* Eqs. 13-14: mass removed per unit volume from a member cell, max(mdot_BH, mdot_Tr) phi dt / V.  With
 * mdot_Tr = (rho - rho_Tr) V / (phi dt) the second candidate is simply rho - rho_Tr (R37: written in that form, which
 * stays finite when phi underflows to 0).  rho, eint are the PRE-step values of the cell. */
static inline double sink_cell_amount(const orc_params *p, const sink_scalars *sc, double r2, double dt, double rho, double eint) {
    double w = exp(-r2 / (sc->r_acc * sc->r_acc));    /* Eq. 9 */
    double phi = w / sc->wsum;                        /* Eq. 11 */
    double V = p->dx * p->dx * p->dx;
    double a = sc->mdot * phi * dt / V;
    double a_tr = rho - rho_truelove(p, rho, eint);   /* Eq. 14 times phi dt / V */
    return a_tr > a ? a_tr : a;
}

static void store_sink_diag(orc_sinks *sk, int64_t s, const sink_scalars *sc) {
    if (sk->rho_inf) sk->rho_inf[s] = sc->rho_inf;
    if (sk->v_inf) sk->v_inf[s] = sc->v_inf;
    if (sk->c_inf) sk->c_inf[s] = sc->c_inf;
    if (sk->r_bh) sk->r_bh[s] = sc->r_bh;
    if (sk->mdot) sk->mdot[s] = sc->mdot;
    if (sk->r_acc) sk->r_acc[s] = sc->r_acc;
    if (sk->wsum) sk->wsum[s] = sc->wsum;
    if (sk->n_member) sk->n_member[s] = sc->n_member;
}

/* ------------------------------------------------------------------------------------------ */
/* Supernova feedback, Sec. 3.2.1                                                               */
/* ------------------------------------------------------------------------------------------ */
typedef struct {
    int64_t ih, jh, kh;
    int g;
    double m_snr, v_snr, vcx, vcy, vcz, e_kin, n_h, r_m, p_rad;
    double pabs[3];           /* error scale only: sum over the stencil of omega rho V |v| per component (the terms of Eq. 18's sum) */
    int regime;
} sn_scalars;

/* omega count (R17): number of the nsub^3 sub-cell centres of cell (i,j,k) with r^2 <= r_K^2 */
static int sn_omega_count(const orc_params *p, double xs, double ys, double zs, int64_t i, int64_t j, int64_t k) {
    const int ns = p->sn_nsub;
    const double rk2 = p->rk_sn * p->rk_sn;
    int cnt = 0;
    for (int qz = 0; qz < ns; ++qz) {
        double ddz = sub_centre(p->x0[2], k, qz, ns, p->dx) - zs;
        for (int qy = 0; qy < ns; ++qy) {
            double ddy = sub_centre(p->x0[1], j, qy, ns, p->dx) - ys;
            for (int qx = 0; qx < ns; ++qx) {
                double ddx = sub_centre(p->x0[0], i, qx, ns, p->dx) - xs;
                if (dist2(ddx, ddy, ddz) <= rk2) cnt += 1;
            }
        }
    }
    return cnt;
}

/* O4: stencil sums, Eq. 18, n_H, R_M, Eqs. 19-20 (R17-R20, R23-R24, R27) */
static void sn_compute_scalars(const orc_params *p, const orc_state *U, double xs, double ys, double zs,
                               double vsx, double vsy, double vsz, double e_sn, double m_ej, sn_scalars *o) {
    const double inv_dx = 1.0 / p->dx;
    const double V = p->dx * p->dx * p->dx;
    const double nsub3 = (double)p->sn_nsub * (double)p->sn_nsub * (double)p->sn_nsub;
    o->ih = host_cell(xs, p->x0[0], inv_dx);
    o->jh = host_cell(ys, p->x0[1], inv_dx);
    o->kh = host_cell(zs, p->x0[2], inv_dx);
    o->g = kernel_halfwidth(p->rk_sn, p->dx);
    const int g = o->g;
    double m_gas = 0.0, px = 0.0, py = 0.0, pz = 0.0, v_snr = 0.0;
    o->pabs[0] = o->pabs[1] = o->pabs[2] = 0.0;
    for (int64_t k = o->kh - g; k <= o->kh + g; ++k)
        for (int64_t j = o->jh - g; j <= o->jh + g; ++j)
            for (int64_t i = o->ih - g; i <= o->ih + g; ++i) {
                int cnt = sn_omega_count(p, xs, ys, zs, i, j, k);
                if (cnt == 0) continue;
                double omega = (double)cnt / nsub3;
                int64_t c = cell_index(p, i, j, k);
                double rho = U->rho[c];
                double vx = U->mx[c] / rho, vy = U->my[c] / rho, vz = U->mz[c] / rho;
                double mcell = omega * rho * V;
                m_gas += mcell;
                px += mcell * vx;
                py += mcell * vy;
                pz += mcell * vz;
                v_snr += omega * V;                                   /* R18 */
                o->pabs[0] += mcell * fabs(vx); o->pabs[1] += mcell * fabs(vy); o->pabs[2] += mcell * fabs(vz);   /* error scale only */
            }
    o->m_snr = m_gas + m_ej;                                          /* L203 */
    o->v_snr = v_snr;
    o->vcx = (px + m_ej * vsx) / o->m_snr;                            /* Eq. 18, R20 */
    o->vcy = (py + m_ej * vsy) / o->m_snr;
    o->vcz = (pz + m_ej * vsz) / o->m_snr;
    o->e_kin = 0.5 * m_ej * ((vsx * vsx + vsy * vsy) + vsz * vsz);    /* L210 */
    o->n_h = o->m_snr / (p->sn_mu_h * o->v_snr);                      /* L203 */
    double m_sf = p->sn_msf_coeff * pow(o->n_h / p->sn_nh_unit, p->sn_msf_exp);
    o->r_m = o->m_snr / m_sf;
    int regime = p->sn_regime;
    if (regime == 0) {                                                /* Eq. 19 */
        if (o->r_m > p->sn_rm_mc) regime = 3;
        else if (o->r_m > p->sn_rm_ej) regime = 2;
        else regime = 1;
    }
    o->regime = regime;
    if (regime == 3) o->p_rad = p->sn_psnr_coeff * pow(o->n_h / p->sn_nh_unit, p->sn_psnr_exp);   /* Eq. 20 */
    else if (regime == 2) o->p_rad = sqrt(2.0 * o->m_snr * p->sn_eps_k * e_sn);                    /* Eq. 19, R23 */
    else o->p_rad = 0.0;                                                                            /* R24 */
}

/* O5: Eq. 17 for one cell with omega > 0 (R21, R22). out = (d rho, d px, d py, d pz, d E). */
static void sn_cell_deposit(const orc_params *p, const sn_scalars *sc, double xs, double ys, double zs,
                            double e_sn, double m_ej, int64_t i, int64_t j, int64_t k, int cnt,
                            double rho, double vx, double vy, double vz, double out[5], double out_abs[5], double out_cond[5]) {
    const double nsub3 = (double)p->sn_nsub * (double)p->sn_nsub * (double)p->sn_nsub;
    double omega = (double)cnt / nsub3;
    double ddx = cell_centre(p->x0[0], i, p->dx) - xs;
    double ddy = cell_centre(p->x0[1], j, p->dx) - ys;
    double ddz = cell_centre(p->x0[2], k, p->dx) - zs;
    double r = sqrt(dist2(ddx, ddy, ddz));
    double rhx = 0.0, rhy = 0.0, rhz = 0.0;
    if (r > 0.0) { rhx = ddx / r; rhy = ddy / r; rhz = ddz / r; }
    double drho = omega * m_ej / sc->v_snr;
    double pscale = (sc->p_rad / sc->v_snr) * omega;                  /* R21 */
    double prx = pscale * rhx, pry = pscale * rhy, prz = pscale * rhz;
    out[0] = drho;
    out[1] = omega * rho * (sc->vcx - vx) + drho * sc->vcx + prx;     /* R22 */
    out[2] = omega * rho * (sc->vcy - vy) + drho * sc->vcy + pry;
    out[3] = omega * rho * (sc->vcz - vz) + drho * sc->vcz + prz;
    out[4] = omega * (e_sn + sc->e_kin) / sc->v_snr + ((sc->vcx * prx + sc->vcy * pry) + sc->vcz * prz);
    /* error scale only (Appendix A; R36): the sum of the absolute values of the TERMS added above, since the
     * velocity-smoothing terms of one particle already cancel against each other */
    out_abs[0] = drho;
    out_abs[1] = omega * rho * (fabs(sc->vcx) + fabs(vx)) + drho * fabs(sc->vcx) + fabs(prx);
    out_abs[2] = omega * rho * (fabs(sc->vcy) + fabs(vy)) + drho * fabs(sc->vcy) + fabs(pry);
    out_abs[3] = omega * rho * (fabs(sc->vcz) + fabs(vz)) + drho * fabs(sc->vcz) + fabs(prz);
    out_abs[4] = omega * (e_sn + sc->e_kin) / sc->v_snr + ((fabs(sc->vcx * prx) + fabs(sc->vcy * pry)) + fabs(sc->vcz * prz));
    /* error scale only: v_COM is known to eps * (number of additions) * pabs / M_snr at best -- the stencil sum of Eq. 18 cancels
     * when the gas already streams away from the particle -- and enters the terms above with these factors */
    out_cond[0] = 0.0;
    out_cond[1] = (omega * rho + drho) * (sc->pabs[0] / sc->m_snr);
    out_cond[2] = (omega * rho + drho) * (sc->pabs[1] / sc->m_snr);
    out_cond[3] = (omega * rho + drho) * (sc->pabs[2] / sc->m_snr);
    out_cond[4] = (fabs(prx) * sc->pabs[0] + fabs(pry) * sc->pabs[1] + fabs(prz) * sc->pabs[2]) / sc->m_snr;
}

static void store_sn_diag(orc_sne *sn, int64_t s, const sn_scalars *sc) {
    if (sn->m_snr) sn->m_snr[s] = sc->m_snr;
    if (sn->v_snr) sn->v_snr[s] = sc->v_snr;
    if (sn->vcx) sn->vcx[s] = sc->vcx;
    if (sn->vcy) sn->vcy[s] = sc->vcy;
    if (sn->vcz) sn->vcz[s] = sc->vcz;
    if (sn->n_h) sn->n_h[s] = sc->n_h;
    if (sn->r_m) sn->r_m[s] = sc->r_m;
    if (sn->p_rad) sn->p_rad[s] = sc->p_rad;
    if (sn->regime) sn->regime[s] = sc->regime;
}

/* ------------------------------------------------------------------------------------------ */
/* Step 3 + Step 5 for one cell (O7).  u = (rho, mx, my, mz, etot, eint) updated in place.      */
/* A = signed accretion sums (6), S = SN sums (5), sn_touched = any SN contributes.             */
/* ------------------------------------------------------------------------------------------ */
static void apply_cell(const orc_params *p, double u[6], const double A[6], const double S[5], int sn_touched,
                       double *eta_out, double *lam_out) {
    /* accretion limiter, Eqs. 15-16: d rho_lim = max[min(d rho, f rho), rho - rho_Tr], generalised by R11 (f, floor) */
    double a = -A[0];
    double eta = 1.0;                                                  /* R12 */
    if (a > 0.0) {
        double alim = a;
        double cap = p->f_max_remove * u[0];
        if (cap < alim) alim = cap;
        double need = u[0] - rho_truelove(p, u[0], u[5]);              /* Eq. 16: never leave the cell above rho_Tr ... */
        if (need > alim) alim = need;
        if (alim > a) alim = a;                                        /* ... but never remove more than was requested */
        double room = u[0] - p->rho_floor;
        if (room < 0.0) room = 0.0;
        if (room < alim) alim = room;
        eta = alim / a;
    }
    for (int f = 0; f < 6; ++f) u[f] = u[f] + eta * A[f];              /* Eq. 6, accretion group */
    double lam = 1.0;
    if (sn_touched) {
        double rho1 = u[0], eint1 = u[5];
        double rho2 = rho1 + S[0];
        double e2 = u[4] + S[4];
        double emin = p->sn_eint_theta * rho2 * (eint1 / rho1);        /* R25 */
        double K = 2.0 * rho2 * (e2 - emin);
        double p1x = u[1], p1y = u[2], p1z = u[3];
        double qx = p1x + S[1], qy = p1y + S[2], qz = p1z + S[3];
        double q2 = (qx * qx + qy * qy) + qz * qz;
        if (!(q2 <= K)) {                                              /* Eq. 21 violated at lambda = 1 */
            double aa = (S[1] * S[1] + S[2] * S[2]) + S[3] * S[3];
            double bb = (p1x * S[1] + p1y * S[2]) + p1z * S[3];
            double cc = ((p1x * p1x + p1y * p1y) + p1z * p1z) - K;
            if (aa > 0.0) {
                double disc = bb * bb - aa * cc;
                if (disc < 0.0) lam = 0.0;
                else {
                    lam = (-bb + sqrt(disc)) / aa;                     /* larger root */
                    if (lam < 0.0) lam = 0.0;
                    if (lam > 1.0) lam = 1.0;
                }
            }
        }
        u[0] = rho2;
        u[1] = p1x + lam * S[1];
        u[2] = p1y + lam * S[2];
        u[3] = p1z + lam * S[3];
        u[4] = e2;
        double ke = ((u[1] * u[1] + u[2] * u[2]) + u[3] * u[3]) / (2.0 * rho2);
        double ei = e2 - ke;                                           /* L241 */
        if (ei < 0.0) ei = 0.0;
        u[5] = ei;
    }
    *eta_out = eta;
    *lam_out = lam;
}

/* ------------------------------------------------------------------------------------------ */
/* Exported: stencil queries (bit-exact membership tests)                                       */
/* ------------------------------------------------------------------------------------------ */

/* Member cells of a sink kernel, unwrapped (i,j,k) triples in (k,j,i) loop order. Returns count. */
int32_t orc_sink_stencil(const orc_params *p, double xs, double ys, double zs, int32_t *ijk_out, int32_t max_cells) {
    const double inv_dx = 1.0 / p->dx;
    int64_t ih = host_cell(xs, p->x0[0], inv_dx), jh = host_cell(ys, p->x0[1], inv_dx), kh = host_cell(zs, p->x0[2], inv_dx);
    int g = kernel_halfwidth(p->rk_sink, p->dx);
    int32_t n = 0;
    for (int64_t k = kh - g; k <= kh + g; ++k)
        for (int64_t j = jh - g; j <= jh + g; ++j)
            for (int64_t i = ih - g; i <= ih + g; ++i) {
                double r2;
                if (!sink_member(p, xs, ys, zs, i, j, k, &r2)) continue;
                if (n < max_cells) { ijk_out[3 * n] = (int32_t)i; ijk_out[3 * n + 1] = (int32_t)j; ijk_out[3 * n + 2] = (int32_t)k; }
                n += 1;
            }
    return n;
}

/* omega counts over the (2g+1)^3 box of an SN, (k,j,i) order; host cell written to host_ijk. Returns box side. */
int32_t orc_sn_omega_box(const orc_params *p, double xs, double ys, double zs, int32_t *counts, int32_t *host_ijk) {
    const double inv_dx = 1.0 / p->dx;
    int64_t ih = host_cell(xs, p->x0[0], inv_dx), jh = host_cell(ys, p->x0[1], inv_dx), kh = host_cell(zs, p->x0[2], inv_dx);
    int g = kernel_halfwidth(p->rk_sn, p->dx);
    int64_t n = 0;
    for (int64_t k = kh - g; k <= kh + g; ++k)
        for (int64_t j = jh - g; j <= jh + g; ++j)
            for (int64_t i = ih - g; i <= ih + g; ++i) counts[n++] = sn_omega_count(p, xs, ys, zs, i, j, k);
    host_ijk[0] = (int32_t)ih; host_ijk[1] = (int32_t)jh; host_ijk[2] = (int32_t)kh;
    return 2 * g + 1;
}

/* ------------------------------------------------------------------------------------------ */
/* Exported: stage functions                                                                    */
/* ------------------------------------------------------------------------------------------ */

static void zero_mesh(double *a, int64_t n) { if (a) memset(a, 0, (size_t)n * sizeof(double)); }

/* Steps 1+2 (O2-O6): fill A, S (must be non-NULL), optional Aabs/Sabs/counts; per-particle diagnostics. */
int orc_deposit(const orc_params *p, const orc_state *U, orc_sinks *sk, orc_sne *sn, double dt, orc_mesh_out *mo) {
    const int64_t N = (int64_t)p->nx * p->ny * p->nz;
    for (int f = 0; f < 6; ++f) { if (!mo->A[f]) return -1; zero_mesh(mo->A[f], N); zero_mesh(mo->Aabs[f], N); }
    for (int f = 0; f < 5; ++f) { if (!mo->S[f]) return -1; zero_mesh(mo->S[f], N); zero_mesh(mo->Sabs[f], N); zero_mesh(mo->Scond[f], N); }
    if (mo->sn_count) memset(mo->sn_count, 0, (size_t)N * sizeof(int32_t));
    if (mo->sink_count) memset(mo->sink_count, 0, (size_t)N * sizeof(int32_t));
    zero_mesh(mo->Tp, N); zero_mesh(mo->Te, N);
    if (2 * kernel_halfwidth(p->rk_sink, p->dx) + 1 > p->nx && sk && sk->n > 0) return -2;   /* R32 */

    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t s = 0; s < (sk ? sk->n : 0); ++s) {
        sink_scalars sc;
        double xs = sk->x[s], ys = sk->y[s], zs = sk->z[s];
        sink_compute_scalars(p, U, xs, ys, zs, sk->vx[s], sk->vy[s], sk->vz[s], sk->m[s], &sc);
        store_sink_diag(sk, s, &sc);
        for (int64_t k = sc.kh - sc.g; k <= sc.kh + sc.g; ++k)
            for (int64_t j = sc.jh - sc.g; j <= sc.jh + sc.g; ++j)
                for (int64_t i = sc.ih - sc.g; i <= sc.ih + sc.g; ++i) {
                    double r2;
                    if (!sink_member(p, xs, ys, zs, i, j, k, &r2)) continue;
                    int64_t c = cell_index(p, i, j, k);
                    double rho = U->rho[c];
                    double a = sink_cell_amount(p, &sc, r2, dt, rho, U->eint[c]);
                    /* Eq. 13 (R1: signed change; R9: same mass fraction from every field) */
                    double d[6];
                    d[0] = -a;
                    d[1] = -a * (U->mx[c] / rho);
                    d[2] = -a * (U->my[c] / rho);
                    d[3] = -a * (U->mz[c] / rho);
                    d[4] = -a * (U->etot[c] / rho);
                    d[5] = -a * (U->eint[c] / rho);
                    /* error scale only (R36): |term| times its condition number with respect to r_acc^2, because
                     * a ~ exp(-r^2/r_acc^2) amplifies a relative change of r_acc^2 by r^2/r_acc^2 (up to 16 r_K^2/dx^2) */
                    double cond = 1.0 + r2 / (sc.r_acc * sc.r_acc);
                    for (int f = 0; f < 6; ++f) {
                        #pragma omp atomic
                        mo->A[f][c] += d[f];
                        if (mo->Aabs[f]) {
                            #pragma omp atomic
                            mo->Aabs[f][c] += fabs(d[f]) * cond;
                        }
                    }
                    if (mo->sink_count) {
                        #pragma omp atomic
                        mo->sink_count[c] += 1;
                    }
                }
    }
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t s = 0; s < (sn ? sn->n : 0); ++s) {
        sn_scalars sc;
        double xs = sn->x[s], ys = sn->y[s], zs = sn->z[s];
        sn_compute_scalars(p, U, xs, ys, zs, sn->vx[s], sn->vy[s], sn->vz[s], sn->e_sn[s], sn->m_ej[s], &sc);
        store_sn_diag(sn, s, &sc);
        for (int64_t k = sc.kh - sc.g; k <= sc.kh + sc.g; ++k)
            for (int64_t j = sc.jh - sc.g; j <= sc.jh + sc.g; ++j)
                for (int64_t i = sc.ih - sc.g; i <= sc.ih + sc.g; ++i) {
                    int cnt = sn_omega_count(p, xs, ys, zs, i, j, k);
                    if (cnt == 0) continue;
                    int64_t c = cell_index(p, i, j, k);
                    double rho = U->rho[c];
                    double d[5], da[5], dc[5];
                    sn_cell_deposit(p, &sc, xs, ys, zs, sn->e_sn[s], sn->m_ej[s], i, j, k, cnt,
                                    rho, U->mx[c] / rho, U->my[c] / rho, U->mz[c] / rho, d, da, dc);
                    for (int f = 0; f < 5; ++f) {
                        #pragma omp atomic
                        mo->S[f][c] += d[f];
                        if (mo->Sabs[f]) {
                            #pragma omp atomic
                            mo->Sabs[f][c] += da[f];
                        }
                        if (mo->Scond[f]) {
                            #pragma omp atomic
                            mo->Scond[f][c] += dc[f];
                        }
                    }
                    if (mo->Tp) {
                        #pragma omp atomic
                        mo->Tp[c] += (fabs(d[1]) + fabs(d[2])) + fabs(d[3]);
                    }
                    if (mo->Te) {
                        #pragma omp atomic
                        mo->Te[c] += fabs(d[4]);
                    }
                    if (mo->sn_count) {
                        #pragma omp atomic
                        mo->sn_count[c] += 1;
                    }
                }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* Appendix A "Particle to buffer mesh", reading R34 of DESIGN.md.          */
/* The paper accumulates E := E + eps |dU^buf| after every addition, r = E / |dU^buf|, and     */
/* clears the N_bit = log2 r + 52 + M least significant mantissa bits.  E as printed depends   */
/* on the order of the additions; we use the order-independent upper bound                      */
/*     E <= eps (k - 1) T,   T = sum_s |dU^s|,  k = number of particles that contributed,      */
/* (every partial sum is <= T in magnitude and the first addition, into zero, is exact), and   */
/* take log2 as the difference of binary exponents rounded up (integer arithmetic only):       */
/*     N_bit = ilogb((k - 1) T) - ilogb(|dU^buf|) + 1 + M,  clamped to [0, 52].                 */
/* k <= 1 or dU^buf == 0: nothing to round.  Clearing bits truncates toward zero.               */
/* ------------------------------------------------------------------------------------------ */
int32_t orc_repro_bits(double x, double T, int32_t k, int32_t M) {
    if (k <= 1 || x == 0.0 || !(T > 0.0)) return 0;
    int nb = ilogb((double)(k - 1) * T) - ilogb(fabs(x)) + 1 + M;
    if (nb < 0) nb = 0;
    if (nb > 52) nb = 52;
    return nb;
}

double orc_repro_round(double x, double T, int32_t k, int32_t M) {
    const int32_t nb = orc_repro_bits(x, T, k, M);
    if (nb == 0) return x;
    uint64_t u;
    memcpy(&u, &x, sizeof(u));
    u &= ~((((uint64_t)1) << nb) - 1);
    memcpy(&x, &u, sizeof(u));
    return x;
}

/* Round the deposited buffers of one step (after orc_deposit, before orc_apply).  Needs Tp, Te and both counts.
 * T is the sum of the magnitudes of the values added to the buffer, one per particle and cell (the paper updates E once
 * per addition of a particle's dU^s, L600-606) -- not of the sub-terms of Eq. 17 that Sabs holds for the test tolerances.
 * Accretion group: the terms of A[0] share a sign, so T = |A[0]|; the other five accretion channels are rebuilt from the
 * rounded A[0] in the rank-one form of R29, A[f] = A[0] U_f / rho, with the PRE-step state U.  SN group: d rho has
 * same-sign terms (T = |S[0]|), d E uses Te, and the three momentum channels share Tp. */
int orc_repro_buffers(const orc_params *p, const orc_state *U, orc_mesh_out *mo, int32_t M) {
    const int64_t N = (int64_t)p->nx * p->ny * p->nz;
    if (!mo->sn_count || !mo->sink_count || !mo->Tp || !mo->Te) return -1;
    for (int64_t c = 0; c < N; ++c) {
        const int32_t kk = mo->sink_count[c], kn = mo->sn_count[c];
        if (kk > 0) {
            const double a0 = orc_repro_round(mo->A[0][c], fabs(mo->A[0][c]), kk, M);
            const double rho = U->rho[c];
            mo->A[0][c] = a0;
            mo->A[1][c] = a0 * (U->mx[c] / rho);
            mo->A[2][c] = a0 * (U->my[c] / rho);
            mo->A[3][c] = a0 * (U->mz[c] / rho);
            mo->A[4][c] = a0 * (U->etot[c] / rho);
            mo->A[5][c] = a0 * (U->eint[c] / rho);
        }
        if (kn > 0) {
            const double Tp = mo->Tp[c];
            mo->S[0][c] = orc_repro_round(mo->S[0][c], fabs(mo->S[0][c]), kn, M);
            mo->S[1][c] = orc_repro_round(mo->S[1][c], Tp, kn, M);
            mo->S[2][c] = orc_repro_round(mo->S[2][c], Tp, kn, M);
            mo->S[3][c] = orc_repro_round(mo->S[3][c], Tp, kn, M);
            mo->S[4][c] = orc_repro_round(mo->S[4][c], mo->Te[c], kn, M);
        }
    }
    return 0;
}

/* Steps 3+5 (O7) on every cell, in place; sn_touched[c] != 0 marks cells with an SN contribution. */
int orc_apply(const orc_params *p, orc_state *U, const orc_mesh_out *mo, const int32_t *sn_touched) {
    const int64_t N = (int64_t)p->nx * p->ny * p->nz;
    #pragma omp parallel for schedule(static)
    for (int64_t c = 0; c < N; ++c) {
        double u[6] = { U->rho[c], U->mx[c], U->my[c], U->mz[c], U->etot[c], U->eint[c] };
        double A[6], S[5];
        for (int f = 0; f < 6; ++f) A[f] = mo->A[f][c];
        for (int f = 0; f < 5; ++f) S[f] = mo->S[f][c];
        double eta, lam;
        apply_cell(p, u, A, S, sn_touched ? sn_touched[c] != 0 : 0, &eta, &lam);
        U->rho[c] = u[0]; U->mx[c] = u[1]; U->my[c] = u[2]; U->mz[c] = u[3]; U->etot[c] = u[4]; U->eint[c] = u[5];
        if (mo->eta) mo->eta[c] = eta;
        if (mo->lam) mo->lam[c] = lam;
    }
    return 0;
}

/* Step 4 (O8, Eq. 5) with the deposition function re-evaluated from the PRE-step state U_old (L79; R15). */
int orc_return(const orc_params *p, const orc_state *U_old, const double *eta, orc_sinks *sk, double dt) {
    const double V = p->dx * p->dx * p->dx;
    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t s = 0; s < sk->n; ++s) {
        sink_scalars sc;
        double xs = sk->x[s], ys = sk->y[s], zs = sk->z[s];
        sink_compute_scalars(p, U_old, xs, ys, zs, sk->vx[s], sk->vy[s], sk->vz[s], sk->m[s], &sc);
        double dm = 0.0, dpx = 0.0, dpy = 0.0, dpz = 0.0, dpabs = 0.0;
        for (int64_t k = sc.kh - sc.g; k <= sc.kh + sc.g; ++k)
            for (int64_t j = sc.jh - sc.g; j <= sc.jh + sc.g; ++j)
                for (int64_t i = sc.ih - sc.g; i <= sc.ih + sc.g; ++i) {
                    double r2;
                    if (!sink_member(p, xs, ys, zs, i, j, k, &r2)) continue;
                    int64_t c = cell_index(p, i, j, k);
                    double rho = U_old->rho[c];
                    double a = sink_cell_amount(p, &sc, r2, dt, rho, U_old->eint[c]);
                    double gain = eta[c] * a * V;                     /* -eta dU^s V, mass */
                    dm += gain;
                    dpx += gain * (U_old->mx[c] / rho);               /* R14 */
                    dpy += gain * (U_old->my[c] / rho);
                    dpz += gain * (U_old->mz[c] / rho);
                    dpabs += gain * ((fabs(U_old->mx[c]) + fabs(U_old->my[c]) + fabs(U_old->mz[c])) / rho);   /* error scale only */
                }
        double m_old = sk->m[s];
        double m_new = m_old + dm;
        if (m_new != 0.0) {                                           /* R43: m = 0 and no gain: velocity undefined by Eq. 5, kept */
            sk->vx[s] = (m_old * sk->vx[s] + dpx) / m_new;            /* u = (m, m v), L49 */
            sk->vy[s] = (m_old * sk->vy[s] + dpy) / m_new;
            sk->vz[s] = (m_old * sk->vz[s] + dpz) / m_new;
        }
        sk->m[s] = m_new;
        if (sk->dm) sk->dm[s] = dm;
        if (sk->dpx) sk->dpx[s] = dpx;
        if (sk->dpy) sk->dpy[s] = dpy;
        if (sk->dpz) sk->dpz[s] = dpz;
        if (sk->dpabs) sk->dpabs[s] = dpabs;
    }
    return 0;
}

/* Eq. 5 for ONE particle from an explicit list of (cell, removed-amount-per-volume) pairs:
 * gain = sum eta[cell] * a * V.  Lets a test feed the worked numbers of Fig. 1 (L83). */
double orc_return_from_list(const double *eta, const int64_t *cells, const double *a, int64_t n, double V) {
    double dm = 0.0;
    for (int64_t q = 0; q < n; ++q) dm += eta[cells[q]] * a[q] * V;
    return dm;
}

/* One whole step: deposit -> (fold = wrap) -> apply -> return.  State and sinks updated in place.
 * scratch_old: 6*N doubles the caller provides for U_old.  mo must hold A, S; sn_count is required when SNe exist. */
int orc_step(const orc_params *p, orc_state *U, orc_sinks *sk, orc_sne *sn, double dt, orc_mesh_out *mo, double *scratch_old) {
    const int64_t N = (int64_t)p->nx * p->ny * p->nz;
    if (!mo->sn_count || !mo->eta) return -1;
    orc_state Uo = { scratch_old, scratch_old + N, scratch_old + 2 * N, scratch_old + 3 * N, scratch_old + 4 * N, scratch_old + 5 * N };
    memcpy(Uo.rho, U->rho, (size_t)N * 8); memcpy(Uo.mx, U->mx, (size_t)N * 8); memcpy(Uo.my, U->my, (size_t)N * 8);
    memcpy(Uo.mz, U->mz, (size_t)N * 8); memcpy(Uo.etot, U->etot, (size_t)N * 8); memcpy(Uo.eint, U->eint, (size_t)N * 8);
    int rc = orc_deposit(p, U, sk, sn, dt, mo);
    if (rc) return rc;
    rc = orc_apply(p, U, mo, mo->sn_count);
    if (rc) return rc;
    if (sk && sk->n > 0) rc = orc_return(p, &Uo, mo->eta, sk, dt);
    return rc;
}

/* ------------------------------------------------------------------------------------------ */
/* Exported: the same definitions evaluated at a LIST of cells only (for grids too large to     */
/* run orc_step on within a test): for each listed (wrapped) cell, sum the contribution of      */
/* every particle whose kernel can reach it, then apply_cell.  Outputs are arrays of length     */
/* n_cells: A (6), S (5), Aabs(6), Sabs(5), eta, lam, new state (6), sn_count.                  */
/* ------------------------------------------------------------------------------------------ */
/* One step with the Appendix A rounding of the buffers between deposit and apply (M = margin bits). */
int orc_step_repro(const orc_params *p, orc_state *U, orc_sinks *sk, orc_sne *sn, double dt, orc_mesh_out *mo,
                   double *scratch_old, int32_t M) {
    const int64_t N = (int64_t)p->nx * p->ny * p->nz;
    if (!mo->sn_count || !mo->eta) return -1;
    orc_state Uo = { scratch_old, scratch_old + N, scratch_old + 2 * N, scratch_old + 3 * N, scratch_old + 4 * N, scratch_old + 5 * N };
    memcpy(Uo.rho, U->rho, (size_t)N * 8); memcpy(Uo.mx, U->mx, (size_t)N * 8); memcpy(Uo.my, U->my, (size_t)N * 8);
    memcpy(Uo.mz, U->mz, (size_t)N * 8); memcpy(Uo.etot, U->etot, (size_t)N * 8); memcpy(Uo.eint, U->eint, (size_t)N * 8);
    int rc = orc_deposit(p, U, sk, sn, dt, mo);
    if (rc) return rc;
    rc = orc_repro_buffers(p, U, mo, M);
    if (rc) return rc;
    rc = orc_apply(p, U, mo, mo->sn_count);
    if (rc) return rc;
    if (sk && sk->n > 0) rc = orc_return(p, &Uo, mo->eta, sk, dt);
    return rc;
}

static inline int64_t periodic_delta(int64_t a, int64_t b, int64_t n) {   /* a - b wrapped to [-n/2, n/2) */
    int64_t d = (a - b) % n;
    if (d < -(n / 2)) d += n;
    if (d >= n - n / 2) d -= n;
    return d;
}

int orc_sample_cells(const orc_params *p, const orc_state *U, const orc_sinks *sk, const orc_sne *sn, double dt,
                     const int64_t *cells, int64_t n_cells,
                     double *A_out, double *S_out, double *Aabs_out, double *Sabs_out,
                     double *eta_out, double *lam_out, double *unew_out, int32_t *sn_count_out) {
    const double inv_dx = 1.0 / p->dx;
    const int gs = kernel_halfwidth(p->rk_sink, p->dx), gn = kernel_halfwidth(p->rk_sn, p->dx);
    for (int64_t q = 0; q < n_cells; ++q) {
        int64_t c = cells[q];
        int64_t ci = c % p->nx, cj = (c / p->nx) % p->ny, ck = c / ((int64_t)p->nx * p->ny);
        double A[6] = {0, 0, 0, 0, 0, 0}, S[5] = {0, 0, 0, 0, 0}, Aa[6] = {0, 0, 0, 0, 0, 0}, Sa[5] = {0, 0, 0, 0, 0};
        int32_t nsn = 0;
        double rho = U->rho[c];
        for (int64_t s = 0; sk && s < sk->n; ++s) {
            int64_t ih = host_cell(sk->x[s], p->x0[0], inv_dx), jh = host_cell(sk->y[s], p->x0[1], inv_dx), kh = host_cell(sk->z[s], p->x0[2], inv_dx);
            int64_t di = periodic_delta(ci, ih, p->nx), dj = periodic_delta(cj, jh, p->ny), dk = periodic_delta(ck, kh, p->nz);
            if (di < -gs || di > gs || dj < -gs || dj > gs || dk < -gs || dk > gs) continue;
            double r2;
            if (!sink_member(p, sk->x[s], sk->y[s], sk->z[s], ih + di, jh + dj, kh + dk, &r2)) continue;
            sink_scalars sc;
            sink_compute_scalars(p, U, sk->x[s], sk->y[s], sk->z[s], sk->vx[s], sk->vy[s], sk->vz[s], sk->m[s], &sc);
            double a = sink_cell_amount(p, &sc, r2, dt, rho, U->eint[c]);
            double d[6] = { -a, -a * (U->mx[c] / rho), -a * (U->my[c] / rho), -a * (U->mz[c] / rho),
                            -a * (U->etot[c] / rho), -a * (U->eint[c] / rho) };
            double cond = 1.0 + r2 / (sc.r_acc * sc.r_acc);
            for (int f = 0; f < 6; ++f) { A[f] += d[f]; Aa[f] += fabs(d[f]) * cond; }
        }
        for (int64_t s = 0; sn && s < sn->n; ++s) {
            int64_t ih = host_cell(sn->x[s], p->x0[0], inv_dx), jh = host_cell(sn->y[s], p->x0[1], inv_dx), kh = host_cell(sn->z[s], p->x0[2], inv_dx);
            int64_t di = periodic_delta(ci, ih, p->nx), dj = periodic_delta(cj, jh, p->ny), dk = periodic_delta(ck, kh, p->nz);
            if (di < -gn || di > gn || dj < -gn || dj > gn || dk < -gn || dk > gn) continue;
            int cnt = sn_omega_count(p, sn->x[s], sn->y[s], sn->z[s], ih + di, jh + dj, kh + dk);
            if (cnt == 0) continue;
            sn_scalars sc;
            sn_compute_scalars(p, U, sn->x[s], sn->y[s], sn->z[s], sn->vx[s], sn->vy[s], sn->vz[s], sn->e_sn[s], sn->m_ej[s], &sc);
            double d[5], da[5], dc[5];
            sn_cell_deposit(p, &sc, sn->x[s], sn->y[s], sn->z[s], sn->e_sn[s], sn->m_ej[s], ih + di, jh + dj, kh + dk, cnt,
                            rho, U->mx[c] / rho, U->my[c] / rho, U->mz[c] / rho, d, da, dc);
            /* the sampled evaluation folds the v_COM conditioning into its one error scale (half the weight of a term) */
            for (int f = 0; f < 5; ++f) { S[f] += d[f]; Sa[f] += da[f] + 0.5 * dc[f]; }
            nsn += 1;
        }
        double u[6] = { U->rho[c], U->mx[c], U->my[c], U->mz[c], U->etot[c], U->eint[c] };
        double eta, lam;
        apply_cell(p, u, A, S, nsn > 0, &eta, &lam);
        for (int f = 0; f < 6; ++f) { A_out[6 * q + f] = A[f]; Aabs_out[6 * q + f] = Aa[f]; unew_out[6 * q + f] = u[f]; }
        for (int f = 0; f < 5; ++f) { S_out[5 * q + f] = S[f]; Sabs_out[5 * q + f] = Sa[f]; }
        eta_out[q] = eta; lam_out[q] = lam; sn_count_out[q] = nsn;
    }
    return 0;
}

/* Per-particle scalars only (no mesh output): used to check sampled particles on large grids. */
int orc_particle_scalars(const orc_params *p, const orc_state *U, orc_sinks *sk, orc_sne *sn) {
    for (int64_t s = 0; sk && s < sk->n; ++s) {
        sink_scalars sc;
        sink_compute_scalars(p, U, sk->x[s], sk->y[s], sk->z[s], sk->vx[s], sk->vy[s], sk->vz[s], sk->m[s], &sc);
        store_sink_diag(sk, s, &sc);
    }
    for (int64_t s = 0; sn && s < sn->n; ++s) {
        sn_scalars sc;
        sn_compute_scalars(p, U, sn->x[s], sn->y[s], sn->z[s], sn->vx[s], sn->vy[s], sn->vz[s], sn->e_sn[s], sn->m_ej[s], &sc);
        store_sn_diag(sn, s, &sc);
    }
    return 0;
}

/* Member cells (wrapped linear indices) and removal amounts a^s_ijk (Eq. 13 mass row, per unit volume) of ONE sink,
 * evaluated from state U; (k,j,i) order.  Returns the member count. */
int32_t orc_sink_amounts(const orc_params *p, const orc_state *U, double xs, double ys, double zs,
                         double vsx, double vsy, double vsz, double ms, double dt,
                         int64_t *cells_out, double *a_out, int32_t max_cells) {
    sink_scalars sc;
    sink_compute_scalars(p, U, xs, ys, zs, vsx, vsy, vsz, ms, &sc);
    int32_t n = 0;
    for (int64_t k = sc.kh - sc.g; k <= sc.kh + sc.g; ++k)
        for (int64_t j = sc.jh - sc.g; j <= sc.jh + sc.g; ++j)
            for (int64_t i = sc.ih - sc.g; i <= sc.ih + sc.g; ++i) {
                double r2;
                if (!sink_member(p, xs, ys, zs, i, j, k, &r2)) continue;
                if (n < max_cells) { cells_out[n] = cell_index(p, i, j, k); const int64_t cc = cell_index(p, i, j, k); a_out[n] = sink_cell_amount(p, &sc, r2, dt, U->rho[cc], U->eint[cc]); }
                n += 1;
            }
    return n;
}

/* ------------------------------------------------------------------------------------------ */
/* Sec. 3.1.2 sink particle creation (readings R38, R39 of DESIGN.md).       */
/* A cell creates a sink if (i) rho > rho_Tr (Eq. 12), (ii) it is a STRICT local density        */
/* maximum among the cells whose centres lie within r_K (rk_sink) of its own, periodic, and     */
/* (iii) the retained accretion buffer is zero there ("forbidding sink particle creation in    */
/* any cell within which dU_ijk is non-zero", L177).  The new sink sits at the cell centre      */
/* with m = (rho - rho_Tr) V and momentum m v; the cell keeps v and its specific energies and   */
/* drops to rho_Tr (L183).  All tests use the state as it is on entry; cells are visited in     */
/* index order, so the output is ordered by cell index.  a0 = accretion d rho^sum (may be       */
/* NULL: no sinks yet).  Returns the number found; at most max_new are written and applied.     */
/* ------------------------------------------------------------------------------------------ */
int64_t orc_create_sinks(const orc_params *p, orc_state *U, const double *a0, int64_t max_new,
                         double *x, double *y, double *z, double *vx, double *vy, double *vz, double *m, int64_t *cells) {
    const int64_t N = (int64_t)p->nx * p->ny * p->nz;
    const double V = p->dx * p->dx * p->dx, rk2 = p->rk_sink * p->rk_sink;
    const int g = kernel_halfwidth(p->rk_sink, p->dx);
    int64_t n = 0;
    unsigned char *flag = (unsigned char *)calloc((size_t)N, 1);
    if (!flag) return -1;
    for (int64_t k = 0; k < p->nz; ++k)
        for (int64_t j = 0; j < p->ny; ++j)
            for (int64_t i = 0; i < p->nx; ++i) {
                const int64_t c = cell_index(p, i, j, k);
                const double rho = U->rho[c];
                if (!(rho > rho_truelove(p, rho, U->eint[c]))) continue;          /* (i)   */
                if (a0 && a0[c] != 0.0) continue;                                  /* (iii) */
                int is_max = 1;
                for (int dk = -g; dk <= g && is_max; ++dk)
                    for (int dj = -g; dj <= g && is_max; ++dj)
                        for (int di = -g; di <= g; ++di) {
                            if (!(di | dj | dk)) continue;
                            const double ox = (double)di * p->dx, oy = (double)dj * p->dx, oz = (double)dk * p->dx;
                            if (dist2(ox, oy, oz) > rk2) continue;
                            if (!(U->rho[cell_index(p, i + di, j + dj, k + dk)] < rho)) { is_max = 0; break; }   /* (ii) */
                        }
                if (is_max) flag[c] = 1;
            }
    for (int64_t c = 0; c < N; ++c) {
        if (!flag[c]) continue;
        if (n < max_new) {
            const int64_t i = c % p->nx, j = (c / p->nx) % p->ny, k = c / ((int64_t)p->nx * p->ny);
            const double rho = U->rho[c], rtr = rho_truelove(p, rho, U->eint[c]);
            const double ms = (rho - rtr) * V, keep = rtr / rho;
            x[n] = cell_centre(p->x0[0], i, p->dx); y[n] = cell_centre(p->x0[1], j, p->dx); z[n] = cell_centre(p->x0[2], k, p->dx);
            vx[n] = U->mx[c] / rho; vy[n] = U->my[c] / rho; vz[n] = U->mz[c] / rho;
            m[n] = ms;
            if (cells) cells[n] = c;
            U->rho[c] = rtr;
            U->mx[c] *= keep; U->my[c] *= keep; U->mz[c] *= keep; U->etot[c] *= keep; U->eint[c] *= keep;
        }
        n += 1;
    }
    free(flag);
    return n;
}

int32_t orc_sizeof_params(void) { return (int32_t)sizeof(orc_params); }

/* threads the timed all-cores build uses (1 in the plain build) */
#ifdef _OPENMP
#include <omp.h>
int32_t orc_threads(void) { return (int32_t)omp_get_max_threads(); }
#else
int32_t orc_threads(void) { return 1; }
#endif
