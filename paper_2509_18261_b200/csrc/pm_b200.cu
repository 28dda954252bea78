// pm_b200.cu -- kernels and C ABI of libpm_b200 (see include/pm.h).  sm_100a only; built with -fmad=false.
//
// Kernels:
//   k_tiles_mark / k_tiles_zero / k_zero_sweep   a0  buffer reset by 8^3 tiles: live tiles from the particle bins, zeroed tile by tile
//                      or, when most of the mesh is live, by a linear sweep (pm_tiles.cuh)
//   k_deposit_sinks    a1-a3  one warp per sink: kernel means -> Bondi-Hoyle rate -> Gaussian weights -> fp64 RED
//   k_deposit_sne      a1,a4,a5  one warp per SN: omega counts -> stencil sums -> Eq. 17 -> fp64 RED (5 channels)
//   k_fold_ghosts      a6  gather fold: every owned cell within g of a face sums its <= 7 ghost images, fixed order
//   k_apply_limited    a7  fused limiter + apply, 128-bit loads/stores, untouched cells skip the state traffic
//   k_return_sinks     a8  one warp per sink: sum eta a V (1, v_old) with a shuffle reduction
//   k_grav_deposit / k_grav_apply / k_grav_kick / k_drift   (f)3  PM gravity: cloud-in-cell deposit (Steps 1, 2, 5),
//                      interpolation + half kick, drift (pm_gravity.cuh)
#include "pm_device.cuh"
#include "pm_tiles.cuh"
#include "pm_fast.cuh"
#include "pm_create.cuh"
#include "pm_gravity.cuh"
#include "pm_slab.cuh"
#include "../../include/pm.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

using namespace pm;

// Preferred shared-memory carve-out (% of the 256 KB L1) of the sink kernels: measured on config 5, 25 / 50 / 75 / 100 %
// give 0.52 / 0.50 / 0.53 / 0.79 ms (deposit) and 0.22 / 0.20 / 0.20 / 0.27 ms (return); the SN kernel is best at the default.
constexpr int kSinkCarveout = 50;
constexpr size_t kSnDenseSmem = (size_t)5 * kAccCells * sizeof(double) + (size_t)kSnDenseWarps * sizeof(SnWarpSmem);

// ---------------------------------------------------------------------------------------------------------------
// context
// ---------------------------------------------------------------------------------------------------------------
// slab memory of a z-slab ctx: send_lo | send_hi | recv_lo | recv_hi | recv_lo' | recv_hi' (the primed pair: odd pm_slab_put steps)
constexpr int kSlabParts = 6;

enum Stage { ST_IDLE = 0, ST_DEPOSITED = 1, ST_FOLDED = 2, ST_APPLIED = 3 };

struct pm_ctx {
    pm_params prm;
    DevP P;
    int device;
    int sm_count;
    cudaStream_t stream;
    double *buf;        // nch * Nb
    double *ret;        // N records of kRetWords doubles (eta, v_old x/y/z): one 32-byte sector per cell (NULL when rk_sink == 0)
    double *ret_tr;     // N: rho_old - rho_Tr where a sink removed mass (Truelove on only; Step 4 re-evaluates Eq. 14 from it)
    double *lam;        // N (debug only)
    double *sink_scal;  // 3 * cap_sinks: mdot, r_acc, sum w
    long long cap_sinks;
    double *dbg_sink;   // 8 * cap
    long long cap_dbg_sink;
    double *dbg_sn;     // 9 * cap
    long long cap_dbg_sn;
    int *err_flag;      // device
    int *err_host;      // pinned
    Stage stage;
    long long n_sinks_dep, n_sne_dep;
    double dt;
    long long launches;
    // host-step staging
    // two slots, so that the upload of one step (host -> device) runs under the download of the one before (device -> host)
    cudaStream_t up_stream, down_stream;
    struct HostSlot {
        double *stg_state;  long long stg_state_cap;
        double *stg_sinks;  long long stg_sinks_cap;
        double *stg_sne;    long long stg_sne_cap;
        cudaEvent_t ev_up, ev_done, ev_down;       // inputs on the device / kernels finished / results on the host
        bool busy;
    } slot[2];
    // particle binning: keys[np] | perm[np] | counts[2*ntile + 1]
    int *bin_mem;       long long bin_cap;
    int *grav_mem;      long long grav_cap;   // the same three arrays for the gravity calls (their own: a kick may come between
                                              // pm_deposit and pm_return_to_particles, which still needs the sink order in bin_mem)
    unsigned char *tile_live; long long ntiles;   // liveness flags of the buffer-mesh tiles (pm_tiles.cuh), rewritten by every pm_deposit
    int nch;            // buffer channels allocated: 6, or 10 with PM_FLAG_REPRODUCIBLE
    bool repro; int repro_M;
    int *create_mem; long long create_cap;   // sink creation scratch: [0] = count, [1 ..] = list
    const double *gperm_x; long long gperm_n; bool gperm_valid;   // gravity: perm in grav_mem orders the n particles at gperm_x by host tile
    bool buffer_valid;  // a deposit + fold has filled the buffer mesh (sink creation reads its accretion channel)
    bool ever_deposited;
    double *slab_mem;   // z-slab mode: send_lo | send_hi | recv_lo | recv_hi, each nch * g * pk doubles (pm_slab.cuh)
    long long slab_elems;   // doubles per slab
    bool slab_packed;   // pm_slab_pack / pm_slab_put has run since the last pm_deposit
    // peer-memory form of the exchange (pm_slab_put): where this rank's two slabs go -- the lower neighbour's recv_hi and the
    // upper neighbour's recv_lo, one pair per step parity (two receive-slab sets, so that a put of step n + 1 never lands in
    // memory the neighbour's fold of step n still reads)
    double *put_lo[2], *put_hi[2];
    void *ipc_base[2];  // bases opened with cudaIpcOpenMemHandle (closed by pm_destroy); NULL when the neighbour is in-process
    bool peers_set;
    bool put_step;      // this step's slabs travelled by pm_slab_put: the fold reads the receive set of put_parity
    int put_parity;
    bool dense_smem_ok; // the device grants the dense SN kernel its shared memory (tile accumulator, 150 KB)
    bool grav_in_ch1;   // buffer channel 1 holds the last pm_gravity_deposit (until the next pm_deposit): the debug view must not
                        // "fill in" its stale tiles
    // pm_step_graph: the four calls of a step captured once into a CUDA graph and replayed while the arguments stay the same
    struct GraphKey { pm_state st; pm_sinks sk; pm_sne sn; double dt; } gkey;
    cudaGraphExec_t gexec;
    cudaStream_t gstream; cudaEvent_t gev_in, gev_out;   // the graph runs on a stream of the ctx's own, ordered against the caller's
                                                        // stream by two events: a default stream cannot be captured
    int gstate;         // 0: nothing; 1: gkey has run once eagerly (scratch memory is in place); 2: gexec replays gkey
    long long glaunches;   // kernels in the graph (pm_launch_count advances by this per replay)
    bool timing;        // PM_FLAG_TIMING
    cudaEvent_t ev[PM_NUM_KERNELS][2];
    bool ev_used[PM_NUM_KERNELS];
    bool force_generic; // PM_FLAG_GENERIC_KERNELS: never take the specialised (g = 3 / n_sub = 4, g = 4) kernels
    char msg[256];
};

// tile flags (one byte per tile) followed, 16-byte aligned, by the two `swept` words of Tiles
static size_t tile_swept_offset(long long ntiles) { return (size_t)((ntiles + 15) & ~15ll); }
static size_t tile_flag_bytes(long long ntiles) { return tile_swept_offset(ntiles) + 16; }

#define PM_FAIL(ctx, code, ...) do { snprintf((ctx)->msg, sizeof((ctx)->msg), __VA_ARGS__); return (code); } while (0)
#define PM_CUDA(ctx, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { \
    snprintf((ctx)->msg, sizeof((ctx)->msg), "%s failed: %s", #call, cudaGetErrorString(e_)); return PM_ECUDA; } } while (0)

static int check_launch(pm_ctx *c, const char *name) {
    cudaError_t e = cudaGetLastError();
    c->launches += 1;
    if (e != cudaSuccess) { snprintf(c->msg, sizeof(c->msg), "launch of %s failed: %s", name, cudaGetErrorString(e)); return PM_ECUDA; }
    return PM_OK;
}

// PM_FLAG_TIMING: events on the launching stream around kernel group k (which = 0 before, 1 after)
static void tick(pm_ctx *c, int k, int which) {
    if (!c->timing) return;
    cudaEventRecord(c->ev[k][which], c->stream);
    if (which) c->ev_used[k] = true;
}

// ---------------------------------------------------------------------------------------------------------------
// a0: buffer reset: see pm_tiles.cuh.  The kernel below is for the test-only views (pm_debug_buffer,
// pm_debug_round_buffers): it stores the zeros that stale tiles stand for and marks them live, so that the raw buffer can be read.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_tiles_materialize(const DevP P, double *__restrict__ buf, const Tiles T, const bool repro,
                                                           const bool keep_n, const int ntiles) {
    const int t = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (t >= ntiles) return;
    const unsigned f = T.live[t];
    const bool lk = f & kLiveK, ln = keep_n || (f & kLiveN);
    unsigned mask = 0;
    if (!lk) mask |= 1u;
    if (!ln) mask |= repro ? 0xFEu : 0x3Eu;
    if (repro && !lk && !ln) mask |= 1u << kChK;
    if (mask) tile_zero(P, buf, t, mask, lane);
    __syncwarp();
    if (lane == 0) T.live[t] = (unsigned char)(f | kLiveK | (keep_n ? 0u : kLiveN));
}

// ---------------------------------------------------------------------------------------------------------------
// a1: host cells -> bins.  Sinks use keys [0, ntile), SNe [ntile, 2 ntile); perm[0..nk) lists sink indices bin by
// bin, perm[nk..nk+nn) SN indices.  Order inside a bin is whatever the atomic append gives (results depend on it
// only through the order of the atomic additions, as they do anyway).
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_bin_count(const DevP P, const double *__restrict__ kx, const double *__restrict__ ky,
                                                   const double *__restrict__ kz, long long nk,
                                                   const double *__restrict__ nx_, const double *__restrict__ ny_,
                                                   const double *__restrict__ nz_, long long nn,
                                                   int *__restrict__ keys, int *__restrict__ counts,
                                                   unsigned char *__restrict__ occ) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= nk + nn) return;
    const bool sink = p < nk;
    const long long q = sink ? p : p - nk;
    const double x = sink ? kx[q] : nx_[q], y = sink ? ky[q] : ny_[q], z = sink ? kz[q] : nz_[q];
    int ih = host_cell(x, P.x0[0], P.inv_dx), jh = host_cell(y, P.x0[1], P.inv_dx), kh = host_cell(z, P.x0[2], P.inv_dx);
    ih = min(max(ih, 0), P.nx - 1); jh = min(max(jh, 0), P.ny - 1); kh = min(max(kh, 0), P.nz - 1);   // outsiders are flagged later
    const int key = bin_key(P, ih, jh, kh) + (sink ? 0 : P.ntile);
    keys[p] = key;
    atomicAdd(counts + key, 1);
    if (occ) occ[key] = 1;            // bin occupancy for the reset (k_tiles_mark)
}

// Exclusive prefix sum of counts[0..n), two levels: every block scans its own 2048 keys in place and publishes its
// total; one block then scans the totals; k_bin_fill adds the block offset back.
constexpr int kScanChunk = 2048;

__global__ void __launch_bounds__(256) k_bin_scan_local(int *__restrict__ counts, int n, int *__restrict__ sums) {
    __shared__ int part[256];
    const int t = threadIdx.x;
    const int base = blockIdx.x * kScanChunk + t * 8;
    int v[8], sum = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { v[i] = (base + i < n) ? counts[base + i] : 0; sum += v[i]; }
    part[t] = sum;
    __syncthreads();
    for (int off = 1; off < 256; off <<= 1) {
        const int add = t >= off ? part[t - off] : 0;
        __syncthreads();
        part[t] += add;
        __syncthreads();
    }
    int run = part[t] - sum;
#pragma unroll
    for (int i = 0; i < 8; ++i) { if (base + i < n) counts[base + i] = run; run += v[i]; }
    if (t == 255) sums[blockIdx.x] = part[255];
}

__global__ void __launch_bounds__(1024) k_bin_scan_sums(int *__restrict__ sums, int n) {
    __shared__ int part[1024];
    const int t = threadIdx.x;
    const int chunk = (n + 1023) / 1024;
    const int lo = min(t * chunk, n), hi = min(lo + chunk, n);
    int sum = 0;
    for (int i = lo; i < hi; ++i) sum += sums[i];
    part[t] = sum;
    __syncthreads();
    for (int off = 1; off < 1024; off <<= 1) {
        const int v = t >= off ? part[t - off] : 0;
        __syncthreads();
        part[t] += v;
        __syncthreads();
    }
    int run = part[t] - sum;
    for (int i = lo; i < hi; ++i) { const int c = sums[i]; sums[i] = run; run += c; }
}

// start[key] (exclusive prefix inside its scan chunk) and sums[chunk] stay as they are, fillc[key] ends as the bin's count: both
// are read again after the fill (dense-bin list, k_deposit_sne_dense)
__global__ void __launch_bounds__(256) k_bin_fill(const int *__restrict__ keys, const int *__restrict__ start, int *__restrict__ fillc,
                                                  const int *__restrict__ sums, int *__restrict__ perm, long long np,
                                                  long long nk) {
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= np) return;
    const int key = keys[p];
    const int pos = start[key] + sums[key / kScanChunk] + atomicAdd(fillc + key, 1);
    perm[pos] = (int)(p < nk ? p : p - nk);
}

// ---------------------------------------------------------------------------------------------------------------
// a1-a3: sinks.  One warp per sink; lanes stride over the (2g+1)^3 box in (k,j,i) order.
// ---------------------------------------------------------------------------------------------------------------
template <bool REPRO>
__global__ void __launch_bounds__(128) k_deposit_sinks(const DevP P, const DevState U, const DevSinks S, const double dt,
                                                       double *__restrict__ buf0, double *__restrict__ scal,
                                                       double *__restrict__ dbg, int *__restrict__ err,
                                                       const int *__restrict__ perm,
                                                       double *__restrict__ ret_tr) {
    const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= S.n) return;
    const long long s = perm[w];
    const double xs = S.x[s], ys = S.y[s], zs = S.z[s];
    const int ih = host_cell(xs, P.x0[0], P.inv_dx), jh = host_cell(ys, P.x0[1], P.inv_dx), kh = host_cell(zs, P.x0[2], P.inv_dx);
    if (ih < 0 || ih >= P.nx || jh < 0 || jh >= P.ny || kh < 0 || kh >= P.nz) {
        if (lane == 0) { atomicOr(err, 1); scal[s] = 0.0; scal[S.n + s] = 1.0; scal[2 * S.n + s] = 1.0; }
        return;
    }
    const double vsx = S.vx[s], vsy = S.vy[s], vsz = S.vz[s], ms = S.m[s];
    const int g = P.gs, B = 2 * g + 1, nc = B * B * B;
    double sum_rho = 0.0, srx = 0.0, sry = 0.0, srz = 0.0, src = 0.0;
    int cnt = 0;
    for (int c = lane; c < nc; c += 32) {
        const int a = c % B, t = c / B, b = t % B, cc = t / B;
        const int i = ih - g + a, j = jh - g + b, k = kh - g + cc;
        const double r2 = dist2(cell_centre(P.x0[0], i, P.dx) - xs, cell_centre(P.x0[1], j, P.dx) - ys,
                                cell_centre(P.x0[2], k, P.dx) - zs);
        if (r2 <= P.rk2_sink) {
            const long long q = owned_index(P, i, j, k);
            const double rho = U.rho[q];
            const double vx = U.mx[q] / rho, vy = U.my[q] / rho, vz = U.mz[q] / rho;
            const double cs = sound_speed(P, rho, U.eint[q]);
            sum_rho += rho;
            srx += rho * (vx - vsx);
            sry += rho * (vy - vsy);
            srz += rho * (vz - vsz);
            src += rho * cs;
            cnt += 1;
        }
    }
    sum_rho = warp_sum(sum_rho); srx = warp_sum(srx); sry = warp_sum(sry); srz = warp_sum(srz); src = warp_sum(src);
    cnt = warp_sum_int(cnt);
    const SinkScalars sc = sink_scalars(P, sum_rho, srx, sry, srz, src, cnt, ms);
    const double ra2 = sc.r_acc * sc.r_acc;
    double wsum = 0.0;
    for (int c = lane; c < nc; c += 32) {
        const int a = c % B, t = c / B, b = t % B, cc = t / B;
        const double r2 = dist2(cell_centre(P.x0[0], ih - g + a, P.dx) - xs, cell_centre(P.x0[1], jh - g + b, P.dx) - ys,
                                cell_centre(P.x0[2], kh - g + cc, P.dx) - zs);
        if (r2 <= P.rk2_sink) wsum += exp(-r2 / ra2);
    }
    wsum = warp_sum(wsum);
    for (int c = lane; c < nc; c += 32) {
        const int a = c % B, t = c / B, b = t % B, cc = t / B;
        const int i = ih - g + a, j = jh - g + b, k = kh - g + cc;
        const double r2 = dist2(cell_centre(P.x0[0], i, P.dx) - xs, cell_centre(P.x0[1], j, P.dx) - ys,
                                cell_centre(P.x0[2], k, P.dx) - zs);
        if (r2 <= P.rk2_sink) {
            double amt = sink_cell_amount(P, r2, sc.r_acc, wsum, sc.mdot, dt);
            if (P.tl_num > 0.0) {                                     // Eqs. 13-14: max(mdot_BH, mdot_Tr) phi dt / V
                const long long q = owned_index(P, i, j, k);
                amt = fmax(amt, truelove_excess(P, U.rho[q], U.eint[q]));
                ret_tr[q] = -CUDART_INF;                              // invalidate last step's entry (rewritten by the apply pass)
            }
            double *dst = buf0 + deposit_index(P, i, j, k);
            red_add(dst, -amt);                                     // R1: signed change
            if (REPRO) red_add(dst + kChK * P.Nb, kSinkUnit);         // Appendix A: contribution count
        }
    }
    if (lane == 0) {
        scal[s] = sc.mdot; scal[S.n + s] = sc.r_acc; scal[2 * S.n + s] = wsum;
        if (dbg) {
            const long long n = S.n;
            dbg[s] = sc.rho_inf; dbg[n + s] = sc.v_inf; dbg[2 * n + s] = sc.c_inf; dbg[3 * n + s] = sc.r_bh;
            dbg[4 * n + s] = sc.mdot; dbg[5 * n + s] = sc.r_acc; dbg[6 * n + s] = wsum; dbg[7 * n + s] = (double)cnt;
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a1, a4, a5: supernovae.  One warp per SN; per-warp shared tables for the omega sub-sampling.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kSnWarps = 8;

template <bool REPRO>
__global__ void __launch_bounds__(kSnWarps * 32) k_deposit_sne(const DevP P, const DevState U, const DevSNe S,
                                                                double *__restrict__ buf, double *__restrict__ dbg,
                                                                int *__restrict__ err, const int *__restrict__ perm) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const long long w = (long long)blockIdx.x * kSnWarps + wib;
    if (w >= S.n) return;
    const long long s = perm[w];
    const int g = P.gn, B = 2 * g + 1, nc = B * B * B;
    const SnTables Tb = sn_tables_at(smem + (size_t)wib * sn_table_bytes(B, P.nsub), B, P.nsub);
    const double xs = S.x[s], ys = S.y[s], zs = S.z[s];
    const int ih = host_cell(xs, P.x0[0], P.inv_dx), jh = host_cell(ys, P.x0[1], P.inv_dx), kh = host_cell(zs, P.x0[2], P.inv_dx);
    if (ih < 0 || ih >= P.nx || jh < 0 || jh >= P.ny || kh < 0 || kh >= P.nz) {
        if (lane == 0) atomicOr(err, 1);
        return;
    }
    sn_fill_tables(P, Tb, lane, xs, ys, zs, ih, jh, kh);
    const double vsx = S.vx[s], vsy = S.vy[s], vsz = S.vz[s], e_sn = S.e_sn[s], m_ej = S.m_ej[s];
    double m_gas = 0.0, px = 0.0, py = 0.0, pz = 0.0, v_snr = 0.0;
    for (int c = lane; c < nc; c += 32) {
        const int a = c % B, t = c / B, b = t % B, cc = t / B;
        const int cnt = sn_omega_count(P, Tb, a, b, cc);
        Tb.cnt[c] = (unsigned short)cnt;
        if (cnt > 0) {
            const double omega = (double)cnt / P.nsub3;
            const long long q = owned_index(P, ih - g + a, jh - g + b, kh - g + cc);
            const double rho = U.rho[q];
            const double vx = U.mx[q] / rho, vy = U.my[q] / rho, vz = U.mz[q] / rho;
            const double mcell = omega * rho * P.V;
            m_gas += mcell;
            px += mcell * vx;
            py += mcell * vy;
            pz += mcell * vz;
            v_snr += omega * P.V;
        }
    }
    m_gas = warp_sum(m_gas); px = warp_sum(px); py = warp_sum(py); pz = warp_sum(pz); v_snr = warp_sum(v_snr);
    const SnScalars sc = sn_scalars(P, m_gas, px, py, pz, v_snr, vsx, vsy, vsz, e_sn, m_ej);
    __syncwarp();
    for (int c = lane; c < nc; c += 32) {
        const int cnt = Tb.cnt[c];
        if (cnt == 0) continue;
        const int a = c % B, t = c / B, b = t % B, cc = t / B;
        const int i = ih - g + a, j = jh - g + b, k = kh - g + cc;
        const long long q = owned_index(P, i, j, k);
        const double rho = U.rho[q];
        double d[5];
        sn_cell_deposit(P, sc, xs, ys, zs, e_sn, m_ej, i, j, k, cnt, rho, U.mx[q] / rho, U.my[q] / rho, U.mz[q] / rho, d);
        double *dst = buf + P.Nb + deposit_index(P, i, j, k);
#pragma unroll
        for (int f = 0; f < 5; ++f) red_add(dst + (long long)f * P.Nb, d[f]);
        if (REPRO) {                                 // Appendix A: error scales and the contribution count (dst is channel 1)
            red_add(dst + (kChTp - 1) * P.Nb, (fabs(d[1]) + fabs(d[2])) + fabs(d[3]));
            red_add(dst + (kChTe - 1) * P.Nb, fabs(d[4]));
            red_add(dst + (kChK - 1) * P.Nb, 1.0);
        }
    }
    if (dbg && lane == 0) {
        const long long n = S.n;
        dbg[s] = sc.m_snr; dbg[n + s] = sc.v_snr; dbg[2 * n + s] = sc.vcx; dbg[3 * n + s] = sc.vcy; dbg[4 * n + s] = sc.vcz;
        dbg[5 * n + s] = sc.n_h; dbg[6 * n + s] = sc.r_m; dbg[7 * n + s] = sc.p_rad; dbg[8 * n + s] = (double)sc.regime;
    }
}

// test-only: stencil of one particle through the same device functions
__global__ void k_debug_stencil(const DevP P, int kind, double xs, double ys, double zs, int *__restrict__ counts,
                                int *__restrict__ host_ijk) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int lane = threadIdx.x & 31;
    const int ih = host_cell(xs, P.x0[0], P.inv_dx), jh = host_cell(ys, P.x0[1], P.inv_dx), kh = host_cell(zs, P.x0[2], P.inv_dx);
    if (lane == 0) { host_ijk[0] = ih; host_ijk[1] = jh; host_ijk[2] = kh; }
    if (kind == 0) {
        const int g = P.gs, B = 2 * g + 1, nc = B * B * B;
        for (int c = lane; c < nc; c += 32) {
            const int a = c % B, t = c / B, b = t % B, cc = t / B;
            const double r2 = dist2(cell_centre(P.x0[0], ih - g + a, P.dx) - xs, cell_centre(P.x0[1], jh - g + b, P.dx) - ys,
                                    cell_centre(P.x0[2], kh - g + cc, P.dx) - zs);
            counts[c] = (r2 <= P.rk2_sink) ? 1 : 0;
        }
    } else {
        const int g = P.gn, B = 2 * g + 1, nc = B * B * B;
        const SnTables T = sn_tables_at(smem, B, P.nsub);
        sn_fill_tables(P, T, lane, xs, ys, zs, ih, jh, kh);
        for (int c = lane; c < nc; c += 32) {
            const int a = c % B, t = c / B, b = t % B, cc = t / B;
            counts[c] = sn_omega_count(P, T, a, b, cc);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a6: ghost fold (gather form).  One thread per owned cell that lies within g of a y or z face; it adds, in the fixed
// order (z image, y image, zy image), the ghost copies of itself to the owned value, for all six channels.  There are no x
// images: the particles wrap x where they add (deposit_index, pm_device.cuh).
// ---------------------------------------------------------------------------------------------------------------
template <int VEC> struct Vec;
template <> struct Vec<1> { typedef double type; };
template <> struct Vec<2> { typedef double2 type; };

template <int VEC>
__device__ __forceinline__ void ldv(const double *p, double v[VEC]) {
    if constexpr (VEC == 2) { const double2 t = *reinterpret_cast<const double2 *>(p); v[0] = t.x; v[1] = t.y; }
    else v[0] = *p;
}
template <int VEC>
__device__ __forceinline__ void stv(double *p, const double v[VEC]) {
    if constexpr (VEC == 2) *reinterpret_cast<double2 *>(p) = make_double2(v[0], v[1]);
    else *p = v[0];
}

// W = 2: one thread folds two x-adjacent cells with 128-bit accesses (needs nx even: every pair is then 16-byte aligned, the
// ghosted row pitch and the x origin gx being even); W = 1 otherwise.  Counts are in units of W cells.
// STAMPS: a stale tile stands for zeros (pm_tiles.cuh) and is not read; an owned cell whose own tile is stale has no live image
// either (a deposit that reaches a ghost cell also claims the tile of its image), so there is nothing to do for it.  Channel 0
// belongs to group K, channels 1..7 to group N, the Appendix A count channel (8) is live where either group is.
// STAMPS = false: plain fold of NCH channels starting at buf (PM gravity, which resets its one channel by a sweep).
// Slab mode (P.zopen): the z images are not in this buffer but in the two slabs received from the z neighbours (Eq. 3 as the
// paper states it: "add the contents of the ghost zones on each rank to the corresponding real zones on other ranks", L67):
// recv_lo = the lower neighbour's HIGH ghost planes, recv_hi = the upper neighbour's LOW ghost planes, each packed as
// [channel][g planes][ny + 2g][row pitch] with stale tiles already replaced by zeros (k_slab_pack).  Same image order, same
// additions: with one rank (its own neighbour) the result is bit-identical to the periodic fold.
template <int W, int NCH, bool STAMPS>
__global__ void __launch_bounds__(256) k_fold_ghosts(const DevP P, double *__restrict__ buf, const Tiles T, long long n_edge,
                                                     long long n_zslab, long long n_yslab, const double *__restrict__ recv_lo,
                                                     const double *__restrict__ recv_hi) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_edge) return;
    const int g = P.g, nx = P.nx, ny = P.ny, nz = P.nz;
    const int nxw = nx / W;
    int i, j, k;
    if (t < n_zslab) {                       // k in [0,g) U [nz-g,nz): full planes
        const long long plane = (long long)nxw * ny;
        int kk = (int)(t / plane);
        long long r = t - (long long)kk * plane;
        j = (int)(r / nxw); i = W * (int)(r - (long long)j * nxw);
        k = kk < g ? kk : nz - 2 * g + kk;
    } else {                                 // interior k, j in [0,g) U [ny-g,ny)   (no x faces: the deposits wrap x themselves)
        long long r = t - n_zslab;
        const long long slab = (long long)nxw * 2 * g;
        int kk = (int)(r / slab);
        r -= (long long)kk * slab;
        int jj = (int)(r / nxw); i = W * (int)(r - (long long)jj * nxw);
        k = g + kk;
        j = jj < g ? jj : ny - 2 * g + jj;
    }
    // image offsets per axis: 0 plus (+n if within g of the low face) or (-n if within g of the high face)
    const int ox = 0;                         // the deposits wrap x themselves (deposit_index): the x ghost columns are empty
    const int oy = j < g ? ny : (j >= ny - g ? -ny : 0);
    const int oz = k < g ? nz : (k >= nz - g ? -nz : 0);
    const long long base = ghost_index(P, i, j, k);
    // images m = 4 cz + 2 cy + cx in ascending order (the fixed order z image, y image, x image); all loads of all channels
    // are issued before any store
    long long img[8];
    bool ok[8];
    unsigned lk = 0xffu, ln = 0xffu;       // bit m: image m's tile is live in group K / N (bit 0: the owned cell's own tile)
    const bool slab = P.zopen != 0;
    const long long slab_ch = (long long)P.g * P.pk;                 // elements of one channel of a received slab
    const double *const rz = oz > 0 ? recv_lo : recv_hi;             // k < g: lower neighbour; k >= nz - g: upper neighbour
    const int pz = oz > 0 ? k : k - (nz - g);                        // plane of the received slab that images plane k
#pragma unroll
    for (int m = 1; m < 8; ++m) {
        const int cx = m & 1, cy = (m >> 1) & 1, cz = m >> 2;
        ok[m] = (!cx || ox) && (!cy || oy) && (!cz || oz);
        img[m] = (slab && cz) ? (long long)pz * P.pk + (long long)(j + cy * oy + P.g) * P.pj + (i + cx * ox + P.gx)
                              : ghost_index(P, i + cx * ox, j + cy * oy, k + cz * oz);
    }
    if (STAMPS && !(tiles_swept(T, 0) && tiles_swept(T, 1))) {
        const bool sk = tiles_swept(T, 0), sn = tiles_swept(T, 1);
        lk = 0; ln = 0;
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            const int cx = m & 1, cy = (m >> 1) & 1, cz = m >> 2;
            if (slab && cz) { if (ok[m]) { lk |= 1u << m; ln |= 1u << m; } continue; }      // received slabs hold values or zeros
            if (m == 0 || ok[m]) {
                const unsigned f = T.live[tile_index(P, i + cx * ox, j + cy * oy, k + cz * oz)];
                lk |= ((f & kLiveK) || sk ? 1u : 0u) << m;
                ln |= ((f & kLiveN) || sn ? 1u : 0u) << m;
            }
        }
        if (!((lk | ln) & 1u)) return;
    }
    double acc[NCH][W];
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        const unsigned live = !STAMPS ? 0xffu : (ch == 0 ? lk : (ch == kChK ? (lk | ln) : ln));
        const double *b = buf + (long long)ch * P.Nb;
        double a[W];
#pragma unroll
        for (int e = 0; e < W; ++e) a[e] = 0.0;
        if (live & 1u) {
            ldv<W>(b + base, a);
#pragma unroll
            for (int m = 1; m < 8; ++m)
                if (ok[m] && (live >> m & 1u)) {
                    double v[W];
                    ldv<W>(((slab && (m >> 2)) ? rz + (long long)ch * slab_ch : b) + img[m], v);
#pragma unroll
                    for (int e = 0; e < W; ++e) a[e] += v[e];
                }
        }
#pragma unroll
        for (int e = 0; e < W; ++e) acc[ch][e] = a[e];
    }
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        const unsigned live = !STAMPS ? 1u : (ch == 0 ? lk : (ch == kChK ? (lk | ln) : ln));
        if (live & 1u) stv<W>(buf + (long long)ch * P.Nb + base, acc[ch]);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Appendix A (PM_FLAG_REPRODUCIBLE): round the six folded buffer channels of every owned cell (repro_round).  The fold
// has already summed the error scales and counts of the ghost images into the owned cell.
// ---------------------------------------------------------------------------------------------------------------
template <int W>
__global__ void __launch_bounds__(256) k_repro_round(const DevP P, double *__restrict__ buf, int M, long long n_items) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n_items) return;
    const int nxw = P.nx / W;
    const int i = W * (int)(t % nxw);
    const long long row = t / nxw;
    const int j = (int)(row % P.ny), k = (int)(row / P.ny);
    double *b = buf + ghost_index(P, i, j, k);
    double ksn[W], ksk[W];
    ldv<W>(b + (long long)kChK * P.Nb, ksn);
#pragma unroll
    for (int e = 0; e < W; ++e) repro_counts(ksn[e], ksn[e], ksk[e]);
    bool any_sn = false, any_sk = false;
#pragma unroll
    for (int e = 0; e < W; ++e) { any_sn |= ksn[e] > 1.0; any_sk |= ksk[e] > 1.0; }
    if (any_sk) {                                                      // same-sign terms: T = |sum|
        double x[W];
        ldv<W>(b, x);
#pragma unroll
        for (int e = 0; e < W; ++e) x[e] = repro_round(x[e], fabs(x[e]), ksk[e], M);
        stv<W>(b, x);
    }
    if (any_sn) {
        double tp[W], te[W], x[W];
        ldv<W>(b + (long long)kChTp * P.Nb, tp);
        ldv<W>(b + (long long)kChTe * P.Nb, te);
#pragma unroll
        for (int f = 1; f <= 5; ++f) {
            ldv<W>(b + (long long)f * P.Nb, x);
#pragma unroll
            for (int e = 0; e < W; ++e) x[e] = repro_round(x[e], f == 1 ? fabs(x[e]) : (f == 5 ? te[e] : tp[e]), ksn[e], M);
            stv<W>(b + (long long)f * P.Nb, x);
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a7: fused limiter + apply.  Each thread owns VEC consecutive cells of one x-row.
// ---------------------------------------------------------------------------------------------------------------
// 128 threads x 6 CTAs per SM: 3.37 ms against 3.44 ms for 256 x 3 (same 80 registers) and 3.96 ms for 256 x 2 (106 registers)
constexpr int kApplyThreads = 128;

template <int VEC, bool LAM, bool TL, bool REPRO>
__global__ void __launch_bounds__(kApplyThreads, 6) k_apply_limited(const DevP P, const DevState U, const double *__restrict__ buf,
                                                       const Tiles T, double *__restrict__ ret, double *__restrict__ ret_tr,
                                                       double *__restrict__ lam_out, const int repro_M,
                                                       unsigned int n_items, unsigned int items_per_row) {
    const unsigned int item_raw = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = item_raw < n_items;
    const unsigned int item = valid ? item_raw : 0u;
    const unsigned int row = item / items_per_row;
    const unsigned int i0 = (item - row * items_per_row) * VEC;
    const unsigned int k = row / (unsigned int)P.ny, j = row - k * (unsigned int)P.ny;
    const long long q = (long long)row * P.nx + i0 + P.zoff;     // state / return-mesh index (zoff: ghost planes of a z slab)
    const long long gq = (long long)(k + P.g) * P.pk + (long long)(j + P.g) * P.pj + (i0 + P.gx);
    // a stale tile stands for zeros and is not read (pm_tiles.cuh); the VEC cells of an item lie in one tile (i0 is even)
    const bool sw_k = tiles_swept(T, 0), sw_n = tiles_swept(T, 1);
    const unsigned lf = (sw_k && sw_n) ? (kLiveK | kLiveN) : __ldg(T.live + tile_index(P, (int)i0, (int)j, (int)k));
    const bool live_k = sw_k || (lf & kLiveK), live_n = sw_n || (lf & kLiveN);
    double b[kBufChannels][VEC];
#pragma unroll
    for (int ch = 0; ch < kBufChannels; ++ch) {
#pragma unroll
        for (int v = 0; v < VEC; ++v) b[ch][v] = 0.0;
        if (ch == 0 ? live_k : live_n) ldv<VEC>(buf + (long long)ch * P.Nb + gq, b[ch]);
    }
    if (REPRO) {   // Appendix A: round the folded sums here, where they are read anyway (rounding never turns a non-zero sum into zero)
        double ksn[VEC], ksk[VEC], tp[VEC], te[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) { ksn[v] = 0.0; tp[v] = 0.0; te[v] = 0.0; }
        if (live_k || live_n) ldv<VEC>(buf + (long long)kChK * P.Nb + gq, ksn);
#pragma unroll
        for (int v = 0; v < VEC; ++v) repro_counts(ksn[v], ksn[v], ksk[v]);
        if (live_n) ldv<VEC>(buf + (long long)kChTp * P.Nb + gq, tp);
        if (live_n) ldv<VEC>(buf + (long long)kChTe * P.Nb + gq, te);
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            b[0][v] = repro_round(b[0][v], fabs(b[0][v]), ksk[v], repro_M);
            b[1][v] = repro_round(b[1][v], fabs(b[1][v]), ksn[v], repro_M);
            b[2][v] = repro_round(b[2][v], tp[v], ksn[v], repro_M);
            b[3][v] = repro_round(b[3][v], tp[v], ksn[v], repro_M);
            b[4][v] = repro_round(b[4][v], tp[v], ksn[v], repro_M);
            b[5][v] = repro_round(b[5][v], te[v], ksn[v], repro_M);
        }
    }
    bool any = false;
#pragma unroll
    for (int ch = 0; ch < kBufChannels; ++ch)
#pragma unroll
        for (int v = 0; v < VEC; ++v) any |= (b[ch][v] != 0.0);
    any = any && valid;
    // Skip at WARP granularity: a warp covers 32*VEC consecutive cells of each field (512 B per stream at VEC = 2), so
    // the state traffic is either whole coalesced lines or nothing (sector-sparse reads waste DRAM bursts).
    // (16- and 8-thread groups, i.e. whole 128- / 64-byte pieces, measured the same 3.41 ms)
    const bool wany = __any_sync(0xffffffffu, any);
    if (LAM && valid && !any) { double one[VEC]; for (int v = 0; v < VEC; ++v) one[v] = 1.0; stv<VEC>(lam_out + (q - P.zoff), one); }
    if (!wany || !valid) return;                // dU^sum = 0 on the whole segment: U unchanged, nothing to read or write
    double *fld[6] = { U.rho, U.mx, U.my, U.mz, U.etot, U.eint };
    double u[6][VEC];
#pragma unroll
    for (int f = 0; f < 6; ++f) ldv<VEC>(fld[f] + q, u[f]);
    double lam[VEC];
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
        double uc[6], bc[6], vold[3] = { 0.0, 0.0, 0.0 };
#pragma unroll
        for (int f = 0; f < 6; ++f) { uc[f] = u[f][v]; bc[f] = b[f][v]; }
        const double exc = (TL && ret_tr) ? truelove_excess(P, uc[0], uc[5]) : 0.0;   // pre-step rho - rho_Tr (Eq. 14), for Step 4
        const double eta = apply_cell<TL>(P, uc, bc, &lam[v], vold);
#pragma unroll
        for (int f = 0; f < 6; ++f) u[f][v] = uc[f];
        if (bc[0] != 0.0 && ret) {              // Step 4 needs eta and the pre-step velocity where a sink removed mass
            double2 *r = reinterpret_cast<double2 *>(ret + 4 * (q + v));      // one whole 32-byte sector per cell
            r[0] = make_double2(eta, vold[0]);
            r[1] = make_double2(vold[1], vold[2]);
            if (TL && ret_tr) ret_tr[q + v] = exc;
        }
    }
    if (!any) return;                           // lanes of a touched segment whose own cells are untouched
#pragma unroll
    for (int f = 0; f < 6; ++f) stv<VEC>(fld[f] + q, u[f]);
    if (LAM) stv<VEC>(lam_out + (q - P.zoff), lam);
}

// ---------------------------------------------------------------------------------------------------------------
// a8: return to particles (Eq. 5).  One warp per sink; shuffle reduction; no atomics.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) k_return_sinks(const DevP P, const DevSinks S, const double dt,
                                                      const double *__restrict__ scal, const double *__restrict__ ret,
                                                      const double *__restrict__ ret_tr,
                                                      const int *__restrict__ perm) {
    const long long w = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (w >= S.n) return;
    const long long s = perm[w];
    const double xs = S.x[s], ys = S.y[s], zs = S.z[s];
    const int ih = host_cell(xs, P.x0[0], P.inv_dx), jh = host_cell(ys, P.x0[1], P.inv_dx), kh = host_cell(zs, P.x0[2], P.inv_dx);
    if (ih < 0 || ih >= P.nx || jh < 0 || jh >= P.ny || kh < 0 || kh >= P.nz) return;   // flagged at deposit
    const double mdot = scal[s], r_acc = scal[S.n + s], wsum = scal[2 * S.n + s];
    const int g = P.gs, B = 2 * g + 1, nc = B * B * B;
    double dm = 0.0, dpx = 0.0, dpy = 0.0, dpz = 0.0;
    for (int c = lane; c < nc; c += 32) {
        const int a = c % B, t = c / B, b = t % B, cc = t / B;
        const int i = ih - g + a, j = jh - g + b, k = kh - g + cc;
        const double r2 = dist2(cell_centre(P.x0[0], i, P.dx) - xs, cell_centre(P.x0[1], j, P.dx) - ys,
                                cell_centre(P.x0[2], k, P.dx) - zs);
        if (r2 <= P.rk2_sink) {
            double amt = sink_cell_amount(P, r2, r_acc, wsum, mdot, dt);
            const long long q = owned_index(P, i, j, k);
            if (ret_tr) amt = fmax(amt, ret_tr[q]);     // Eq. 14 re-evaluated from the pre-step rho - rho_Tr kept by the apply pass
            if (amt > 0.0) {                     // amt == 0 deposits nothing, so the return mesh has no entry there
                const double2 r0 = reinterpret_cast<const double2 *>(ret + 4 * q)[0], r1 = reinterpret_cast<const double2 *>(ret + 4 * q)[1];
                const double gain = r0.x * amt * P.V;
                dm += gain;
                dpx += gain * r0.y;
                dpy += gain * r1.x;
                dpz += gain * r1.y;
            }
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

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
static int ceil_div_pos(double a, double b) { return (int)std::ceil(a / b); }

static bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

static int grow(pm_ctx *c, double **p, long long *cap, long long need) {
    if (need <= *cap) return PM_OK;
    c->gstate = 0;                          // a captured step (pm_step_graph) holds the old address
    if (*p) { PM_CUDA(c, cudaFree(*p)); *p = nullptr; *cap = 0; }
    long long n = need + need / 4 + 64;
    cudaError_t e = cudaMalloc(p, (size_t)n * sizeof(double));
    if (e != cudaSuccess) { *p = nullptr; PM_FAIL(c, PM_ENOMEM, "cudaMalloc of %lld doubles failed: %s", n, cudaGetErrorString(e)); }
    *cap = n;
    return PM_OK;
}

extern "C" int pm_create(const pm_params *prm, int device, void *cuda_stream, pm_ctx **out) {
    if (!prm || !out) return PM_EINVAL;
    *out = nullptr;
    if (prm->nx < 1 || prm->ny < 1 || prm->nz < 1 || !(prm->dx > 0.0)) return PM_EINVAL;
    if (prm->rk_sink < 0.0 || prm->rk_sn < 0.0) return PM_EINVAL;
    if (prm->rk_sn > 0.0 && (prm->sn_nsub < 1 || prm->sn_nsub > 8)) return PM_EINVAL;
    if (prm->sn_regime < 0 || prm->sn_regime > 3) return PM_EINVAL;
    if (!(prm->f_max_remove >= 0.0 && prm->f_max_remove <= 1.0) || prm->rho_floor < 0.0) return PM_EINVAL;
    if (!(prm->truelove_J >= 0.0) || (prm->truelove_J > 0.0 && !(prm->G > 0.0))) return PM_EINVAL;
    const int gs = prm->rk_sink > 0.0 ? ceil_div_pos(prm->rk_sink, prm->dx) : 0;
    const int gn = prm->rk_sn > 0.0 ? ceil_div_pos(prm->rk_sn, prm->dx) : 0;
    const int g = gs > gn ? gs : gn;
    if (g < 1 || g > 8) return PM_EINVAL;
    if (prm->nx < 2 * g + 1 || prm->ny < 2 * g + 1 || prm->nz < 2 * g + 1) return PM_EINVAL;     // R32
    const long long N = (long long)prm->nx * prm->ny * prm->nz;
    if (prm->z_slab != 0 && prm->z_slab != 1) return PM_EINVAL;
    if ((long long)prm->nx * prm->ny * (prm->nz + (prm->z_slab ? 2 * g : 0)) >= (1ll << 31)) return PM_EINVAL;
    if ((long long)(prm->nx + 2 * g + 2) * (prm->ny + 2 * g) * (prm->nz + 2 * g) >= (1ll << 31)) return PM_EINVAL;

    pm_ctx *c = new (std::nothrow) pm_ctx();
    if (!c) return PM_ENOMEM;
    std::memset(c, 0, sizeof(*c));
    c->prm = *prm;
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    DevP &P = c->P;
    P.nx = prm->nx; P.ny = prm->ny; P.nz = prm->nz;
    P.g = g; P.gs = gs; P.gn = gn; P.nsub = prm->sn_nsub > 0 ? prm->sn_nsub : 1; P.regime = prm->sn_regime;
    P.gx = (g + 1) & ~1;
    P.pj = prm->nx + 2 * P.gx; P.pk = P.pj * (prm->ny + 2 * g);
    P.N = N; P.Nb = P.pk * (prm->nz + 2 * g);
    P.dx = prm->dx; P.inv_dx = 1.0 / prm->dx; P.V = prm->dx * prm->dx * prm->dx;
    for (int a = 0; a < 3; ++a) P.x0[a] = prm->x0[a];
    P.G = prm->G; P.gamma = prm->gamma; P.cs_iso = prm->cs_iso;
    P.rk_sink = prm->rk_sink; P.rk2_sink = prm->rk_sink * prm->rk_sink;
    P.rk_sn = prm->rk_sn; P.rk2_sn = prm->rk_sn * prm->rk_sn;
    P.lambda = prm->bondi_lambda; P.fmax = prm->f_max_remove; P.rho_floor = prm->rho_floor;
    P.eps_k = prm->sn_eps_k; P.rm_ej = prm->sn_rm_ej; P.rm_mc = prm->sn_rm_mc;
    P.msf_c = prm->sn_msf_coeff; P.msf_e = prm->sn_msf_exp; P.psnr_c = prm->sn_psnr_coeff; P.psnr_e = prm->sn_psnr_exp;
    P.mu_h = prm->sn_mu_h; P.nh_unit = prm->sn_nh_unit; P.theta = prm->sn_eint_theta;
    P.tl_num = prm->truelove_J * prm->truelove_J * 3.14159265358979323846; P.tl_den = prm->G * prm->dx * prm->dx;
    P.nsub3 = (double)P.nsub * (double)P.nsub * (double)P.nsub;
    const int sbm = (1 << kSbLog2) - 1;
    P.nsbx = (((prm->nx + 7) >> 3) + sbm) >> kSbLog2; P.nsby = (((prm->ny + 7) >> 3) + sbm) >> kSbLog2; P.nsbz = (((prm->nz + 7) >> 3) + sbm) >> kSbLog2;
    P.ntile = (P.nsbx * P.nsby * P.nsbz) << (3 * kSbLog2);
    P.ntx = ((prm->nx + g + 7) >> 3) + 1; P.nty = ((prm->ny + g + 7) >> 3) + 1; P.ntz = ((prm->nz + g + 7) >> 3) + 1;
    c->ntiles = (long long)P.ntx * P.nty * P.ntz;
    P.zopen = prm->z_slab; P.zoff = prm->z_slab ? g * prm->ny * prm->nx : 0;

    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess) {   // L1 / shared-memory split of the particle kernels (measured)
        e = cudaFuncSetAttribute(k_deposit_sinks_g4<false, false>, cudaFuncAttributePreferredSharedMemoryCarveout, kSinkCarveout);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_deposit_sinks_g4<true, false>, cudaFuncAttributePreferredSharedMemoryCarveout, kSinkCarveout);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_deposit_sinks_g4<false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, kSinkCarveout);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_deposit_sinks_g4<true, true>, cudaFuncAttributePreferredSharedMemoryCarveout, kSinkCarveout);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_return_sinks_g4, cudaFuncAttributePreferredSharedMemoryCarveout, kSinkCarveout);
    }
    if (e == cudaSuccess) {
        c->dense_smem_ok = cudaFuncSetAttribute(k_deposit_sne_dense, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSnDenseSmem) == cudaSuccess;
        cudaGetLastError();
    }
    c->repro = (prm->flags & PM_FLAG_REPRODUCIBLE) != 0;
    c->repro_M = 28;                                  // the paper's example margin (L612)
    c->nch = c->repro ? kReproChannels : kBufChannels;
    if (e == cudaSuccess) e = cudaMalloc(&c->buf, (size_t)c->nch * P.Nb * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&c->tile_live, tile_flag_bytes(c->ntiles));
    // before the first deposit every tile is stale = zeros
    if (e == cudaSuccess) e = cudaMemsetAsync(c->tile_live, 0, tile_flag_bytes(c->ntiles), c->stream);
    const long long Nst = N + 2ll * P.zoff;              // cells of a state array / of the return mesh (z ghost planes in slab mode)
    if (e == cudaSuccess && gs > 0) e = cudaMalloc(&c->ret, (size_t)kRetWords * Nst * sizeof(double));
    if (e == cudaSuccess && gs > 0 && P.tl_num > 0.0) e = cudaMalloc(&c->ret_tr, (size_t)Nst * sizeof(double));
    if (e == cudaSuccess && P.zopen) {
        c->slab_elems = (long long)c->nch * g * P.pk;
        e = cudaMalloc(&c->slab_mem, (size_t)kSlabParts * c->slab_elems * sizeof(double));
        if (e == cudaSuccess) e = cudaMemsetAsync(c->slab_mem, 0, (size_t)kSlabParts * c->slab_elems * sizeof(double), c->stream);
    }
    if (e == cudaSuccess && (prm->flags & PM_FLAG_DEBUG_LAMBDA)) e = cudaMalloc(&c->lam, (size_t)N * sizeof(double));
    if (e == cudaSuccess) e = cudaMalloc(&c->err_flag, sizeof(int));
    if (e == cudaSuccess) e = cudaMallocHost(&c->err_host, 2 * sizeof(int));   // [0] error flag, [1] sink-creation count
    if (e == cudaSuccess) e = cudaMemsetAsync(c->err_flag, 0, sizeof(int), c->stream);
    if (e == cudaSuccess && c->ret) e = cudaMemsetAsync(c->ret, 0, (size_t)kRetWords * Nst * sizeof(double), c->stream);
    if (e == cudaSuccess) {
        // opt in to the dynamic shared memory the SN kernel may need (<= 8 warps x tables)
        const size_t smem = kSnWarps * sn_table_bytes(2 * (gn > 0 ? gn : 1) + 1, P.nsub);
        if (smem > 48 * 1024) e = cudaFuncSetAttribute(k_deposit_sne<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess && smem > 48 * 1024) e = cudaFuncSetAttribute(k_deposit_sne<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    }
    if (e != cudaSuccess) {
        int rc = (e == cudaErrorMemoryAllocation) ? PM_ENOMEM : PM_ECUDA;
        cudaGetLastError();
        if (c->buf) cudaFree(c->buf);
        if (c->tile_live) cudaFree(c->tile_live);
        if (c->slab_mem) cudaFree(c->slab_mem);
        if (c->ret) cudaFree(c->ret);
        if (c->ret_tr) cudaFree(c->ret_tr);
        if (c->lam) cudaFree(c->lam);
        if (c->err_flag) cudaFree(c->err_flag);
        if (c->err_host) cudaFreeHost(c->err_host);
        delete c;
        return rc;
    }
    c->force_generic = (prm->flags & PM_FLAG_GENERIC_KERNELS) != 0;
    c->timing = (prm->flags & PM_FLAG_TIMING) != 0;
    if (c->timing)
        for (int k = 0; k < PM_NUM_KERNELS; ++k) { cudaEventCreate(&c->ev[k][0]); cudaEventCreate(&c->ev[k][1]); }
    c->stage = ST_IDLE;
    *out = c;
    return PM_OK;
}

extern "C" int pm_destroy(pm_ctx *c) {
    if (!c) return PM_EINVAL;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    double *ptrs[] = { c->buf, c->ret, c->ret_tr, c->lam, c->sink_scal, c->dbg_sink, c->dbg_sn, c->slot[0].stg_state, c->slot[0].stg_sinks,
                       c->slot[0].stg_sne, c->slot[1].stg_state, c->slot[1].stg_sinks, c->slot[1].stg_sne };
    for (double *p : ptrs) if (p) cudaFree(p);
    if (c->timing)
        for (int k = 0; k < PM_NUM_KERNELS; ++k) { cudaEventDestroy(c->ev[k][0]); cudaEventDestroy(c->ev[k][1]); }
    if (c->gexec) cudaGraphExecDestroy(c->gexec);
    if (c->gstream) { cudaStreamSynchronize(c->gstream); cudaStreamDestroy(c->gstream); cudaEventDestroy(c->gev_in); cudaEventDestroy(c->gev_out); }
    if (c->up_stream) {
        cudaStreamSynchronize(c->up_stream); cudaStreamSynchronize(c->down_stream);
        cudaStreamDestroy(c->up_stream); cudaStreamDestroy(c->down_stream);
        for (int k = 0; k < 2; ++k) { cudaEventDestroy(c->slot[k].ev_up); cudaEventDestroy(c->slot[k].ev_done); cudaEventDestroy(c->slot[k].ev_down); }
    }
    if (c->bin_mem) cudaFree(c->bin_mem);
    if (c->grav_mem) cudaFree(c->grav_mem);
    if (c->tile_live) cudaFree(c->tile_live);
    for (int k = 0; k < 2; ++k) if (c->ipc_base[k] && !(k == 1 && c->ipc_base[1] == c->ipc_base[0])) cudaIpcCloseMemHandle(c->ipc_base[k]);
    if (c->slab_mem) cudaFree(c->slab_mem);
    if (c->create_mem) cudaFree(c->create_mem);
    if (c->err_flag) cudaFree(c->err_flag);
    if (c->err_host) cudaFreeHost(c->err_host);
    delete c;
    return PM_OK;
}

extern "C" int pm_set_repro_margin(pm_ctx *c, int32_t M) {
    if (!c) return PM_EINVAL;
    if (!c->repro) PM_FAIL(c, PM_EINVAL, "pm_set_repro_margin needs PM_FLAG_REPRODUCIBLE");
    if (M < 0 || M > 52) PM_FAIL(c, PM_EINVAL, "pm_set_repro_margin: M must be in [0, 52]");
    c->repro_M = M;
    c->gstate = 0;       // the margin is an argument of the captured apply kernel
    return PM_OK;
}

extern "C" const char *pm_last_error(const pm_ctx *c) { return c ? c->msg : "null ctx"; }
extern "C" int64_t pm_launch_count(const pm_ctx *c) { return c ? c->launches : 0; }

static Tiles tiles_of(const pm_ctx *c) { return Tiles{ c->tile_live, reinterpret_cast<int *>(c->tile_live + tile_swept_offset(c->ntiles)) }; }

static bool state_ok(const pm_state *s) { return s && s->rho && s->mx && s->my && s->mz && s->etot && s->eint; }

extern "C" int pm_deposit(pm_ctx *c, const pm_state *st, const pm_sinks *sk, const pm_sne *sn, double dt) {
    if (!c) return PM_EINVAL;
    if (!state_ok(st)) PM_FAIL(c, PM_EINVAL, "pm_deposit: null state pointer");
    const long long nk = sk ? sk->n : 0, nn = sn ? sn->n : 0;
    if (nk < 0 || nn < 0) PM_FAIL(c, PM_EINVAL, "pm_deposit: negative particle count");
    if (nk > 0 && c->P.gs == 0) PM_FAIL(c, PM_EINVAL, "pm_deposit: sinks given but rk_sink == 0");
    if (nn > 0 && c->P.gn == 0) PM_FAIL(c, PM_EINVAL, "pm_deposit: SNe given but rk_sn == 0");
    if (nk > 0 && !(sk->x && sk->y && sk->z && sk->vx && sk->vy && sk->vz && sk->m)) PM_FAIL(c, PM_EINVAL, "pm_deposit: null sink array");
    if (nn > 0 && !(sn->x && sn->y && sn->z && sn->vx && sn->vy && sn->vz && sn->e_sn && sn->m_ej)) PM_FAIL(c, PM_EINVAL, "pm_deposit: null SN array");
    PM_CUDA(c, cudaSetDevice(c->device));
    const DevP &P = c->P;
    const bool dbg = (c->prm.flags & PM_FLAG_DEBUG_SCALARS) != 0;
    int rc;
    if ((rc = grow(c, &c->sink_scal, &c->cap_sinks, 3 * nk)) != PM_OK) return rc;
    if (dbg && (rc = grow(c, &c->dbg_sink, &c->cap_dbg_sink, 8 * nk)) != PM_OK) return rc;
    if (dbg && (rc = grow(c, &c->dbg_sn, &c->cap_dbg_sn, 9 * nn)) != PM_OK) return rc;

    for (int k = 0; k < PM_NUM_KERNELS; ++k) c->ev_used[k] = false;
    const long long np = nk + nn;
    int *keys = nullptr, *perm = nullptr, *counts = nullptr, *sums = nullptr, *live = nullptr, *fillc = nullptr, *dense_n = nullptr, *dense_list = nullptr;
    unsigned char *occ = nullptr;
    if (np > 0 || P.zopen) {   // a1: bin particles by host tile (a slab without particles still needs the scratch of the reset)
        if (np >= (1ll << 31)) PM_FAIL(c, PM_EINVAL, "pm_deposit: too many particles");
        const int nkeys = 2 * P.ntile + 1;
        const int nscan = (nkeys + kScanChunk - 1) / kScanChunk;
        const int nocc = (2 * P.ntile + 3) / 4;                         // bin occupancy bytes, in ints
        // keys | perm | start (counts, then their scan) | chunk sums | fill counters | occupancy | live-tile counters (2) |
        // dense-bin counters (front, back, queue head) | dense-bin list
        const long long need = 2 * np + nkeys + nscan + nkeys + nocc + 2 + 3 + P.ntile;
        if (need > c->bin_cap) {
            c->gstate = 0;                  // a captured step (pm_step_graph) holds the old address
            if (c->bin_mem) { PM_CUDA(c, cudaFree(c->bin_mem)); c->bin_mem = nullptr; c->bin_cap = 0; }
            const long long cap = need + need / 4;
            cudaError_t e = cudaMalloc(&c->bin_mem, (size_t)cap * sizeof(int));
            if (e != cudaSuccess) { c->bin_mem = nullptr; PM_FAIL(c, PM_ENOMEM, "cudaMalloc of bins failed: %s", cudaGetErrorString(e)); }
            c->bin_cap = cap;
        }
        keys = c->bin_mem; perm = keys + np; counts = perm + np;
        sums = counts + nkeys;
        fillc = sums + nscan;
        occ = reinterpret_cast<unsigned char *>(fillc + nkeys);
        live = fillc + nkeys + nocc;
        dense_n = live + 2;
        dense_list = dense_n + 3;
        PM_CUDA(c, cudaMemsetAsync(counts, 0, (size_t)(nkeys + nscan + nkeys + nocc + 2 + 3) * sizeof(int), c->stream));
        if (np > 0) {
            const unsigned blocks = (unsigned)((np + 255) / 256);
            tick(c, PM_K_BIN, 0);
            k_bin_count<<<blocks, 256, 0, c->stream>>>(P, nk ? sk->x : nullptr, nk ? sk->y : nullptr, nk ? sk->z : nullptr, nk,
                                                       nn ? sn->x : nullptr, nn ? sn->y : nullptr, nn ? sn->z : nullptr, nn, keys, counts, occ);
            if ((rc = check_launch(c, "k_bin_count")) != PM_OK) return rc;
            k_bin_scan_local<<<nscan, 256, 0, c->stream>>>(counts, nkeys, sums);
            if ((rc = check_launch(c, "k_bin_scan_local")) != PM_OK) return rc;
            k_bin_scan_sums<<<1, 1024, 0, c->stream>>>(sums, nscan);
            if ((rc = check_launch(c, "k_bin_scan_sums")) != PM_OK) return rc;
            k_bin_fill<<<blocks, 256, 0, c->stream>>>(keys, counts, fillc, sums, perm, np, nk);
            if ((rc = check_launch(c, "k_bin_fill")) != PM_OK) return rc;
            tick(c, PM_K_BIN, 1);
        }
    }
    // a0: reset (L59 "all cells initialized to zero").  The tiles this step's particles can add into are marked live (from the
    // bin occupancy) and zeroed; all others are stale and taken as zeros by the readers (pm_tiles.cuh).
    if (np == 0 && !P.zopen) PM_CUDA(c, cudaMemsetAsync(c->tile_live, 0, tile_flag_bytes(c->ntiles), c->stream));   // flags and `swept`
    if (np > 0 || P.zopen) {
        const Tiles T = tiles_of(c);
        tick(c, PM_K_ZERO, 0);
        k_tiles_mark<<<(unsigned)((c->ntiles + 255) / 256), 256, 0, c->stream>>>(P, T, occ, (int)c->ntiles, nk > 0, nn > 0, live);
        if ((rc = check_launch(c, "k_tiles_mark")) != PM_OK) return rc;
        const unsigned zblocks = (unsigned)std::min<long long>((c->ntiles + 7) / 8, (long long)c->sm_count * 16);
        k_tiles_zero<<<zblocks, 256, 0, c->stream>>>(P, c->buf, T, c->repro, (int)c->ntiles, live);
        if ((rc = check_launch(c, "k_tiles_zero")) != PM_OK) return rc;
        k_zero_sweep<<<c->sm_count * 16, 256, 0, c->stream>>>(P, c->buf, c->repro, (int)c->ntiles, live, T.swept);
        if ((rc = check_launch(c, "k_zero_sweep")) != PM_OK) return rc;
        tick(c, PM_K_ZERO, 1);
    }
    const DevState U = { st->rho, st->mx, st->my, st->mz, st->etot, st->eint };
    if (nk > 0) {
        const DevSinks S = { nk, sk->x, sk->y, sk->z, sk->vx, sk->vy, sk->vz, sk->m, sk->dm, sk->dpx, sk->dpy, sk->dpz };
        const unsigned blocks = (unsigned)((nk + 3) / 4);
        tick(c, PM_K_SINKS, 0);
        if (P.gs == 4 && !c->force_generic)
            (P.tl_num > 0.0 ? (c->repro ? k_deposit_sinks_g4<true, true> : k_deposit_sinks_g4<false, true>)
                            : (c->repro ? k_deposit_sinks_g4<true, false> : k_deposit_sinks_g4<false, false>))<<<blocks, kFastSinkWarps * 32, 0, c->stream>>>(P, U, S, dt, c->buf, c->sink_scal, dbg ? c->dbg_sink : nullptr, c->err_flag, perm, c->ret_tr);
        else
            (c->repro ? k_deposit_sinks<true> : k_deposit_sinks<false>)<<<blocks, 128, 0, c->stream>>>(P, U, S, dt, c->buf, c->sink_scal, dbg ? c->dbg_sink : nullptr, c->err_flag, perm, c->ret_tr);
        if ((rc = check_launch(c, "k_deposit_sinks")) != PM_OK) return rc;
        tick(c, PM_K_SINKS, 1);
    }
    if (nn > 0) {
        const DevSNe S = { nn, sn->x, sn->y, sn->z, sn->vx, sn->vy, sn->vz, sn->e_sn, sn->m_ej };
        const unsigned blocks = (unsigned)((nn + kSnWarps - 1) / kSnWarps);
        const size_t smem = kSnWarps * sn_table_bytes(2 * P.gn + 1, P.nsub);
        tick(c, PM_K_SNE, 0);
        if (P.gn == 3 && P.nsub == 4 && !c->force_generic && 7 * P.pk < (1ll << 31)) {   // box offsets are 32-bit there
            // bins with many particles go through the shared-memory tile accumulator (pm_sn_fast.cuh), the others add directly
            // (opt-in, PM_FLAG_SMEM_TILES: measured slower than the direct path at every threshold on B200)
            const bool dense = !c->repro && c->dense_smem_ok && (c->prm.flags & PM_FLAG_SMEM_TILES) != 0;
            const int *keys_sn = keys + nk, *cnt_sn = dense ? fillc + P.ntile : nullptr;
            if (dense) {
                k_sn_dense_bins<<<(unsigned)((P.ntile + 255) / 256), 256, 0, c->stream>>>(P.ntile, cnt_sn, dense_list, dense_n);
                if ((rc = check_launch(c, "k_sn_dense_bins")) != PM_OK) return rc;
            }
            (c->repro ? k_deposit_sne_g3n4<true> : k_deposit_sne_g3n4<false>)<<<(unsigned)((nn + kFastSnWarps - 1) / kFastSnWarps), kFastSnWarps * 32, 0, c->stream>>>(P, U, S, c->buf, dbg ? c->dbg_sn : nullptr, c->err_flag, perm + nk, keys_sn, cnt_sn, kSnDenseMin);
            if (dense) {
                if ((rc = check_launch(c, "k_deposit_sne_g3n4")) != PM_OK) return rc;
                k_deposit_sne_dense<<<c->sm_count, kSnDenseWarps * 32, kSnDenseSmem, c->stream>>>(P, U, S, c->buf, dbg ? c->dbg_sn : nullptr, c->err_flag, perm + nk,
                                                                                               counts, sums, cnt_sn, dense_list, dense_n, dense_n + 2, kScanChunk, (int)nk);
            }
        } else
            (c->repro ? k_deposit_sne<true> : k_deposit_sne<false>)<<<blocks, kSnWarps * 32, smem, c->stream>>>(P, U, S, c->buf, dbg ? c->dbg_sn : nullptr, c->err_flag, perm + nk);
        if ((rc = check_launch(c, "k_deposit_sne")) != PM_OK) return rc;
        tick(c, PM_K_SNE, 1);
    }
    c->n_sinks_dep = nk; c->n_sne_dep = nn; c->dt = dt;
    c->ever_deposited = true;
    c->grav_in_ch1 = false;
    c->slab_packed = false;
    c->put_step = false;
    c->stage = ST_DEPOSITED;
    c->buffer_valid = false;              // unfolded until pm_fold_ghosts
    return PM_OK;
}

extern "C" int pm_fold_ghosts(pm_ctx *c) {
    if (!c) return PM_EINVAL;
    if (c->stage != ST_DEPOSITED) PM_FAIL(c, PM_EORDER, "pm_fold_ghosts must follow pm_deposit");
    PM_CUDA(c, cudaSetDevice(c->device));
    const DevP &P = c->P;
    const long long g2 = 2 * P.g;
    const int W = P.nx % 2 == 0 ? 2 : 1;
    const long long n_z = g2 * P.ny * P.nx / W;
    const long long n_y = (long long)(P.nz - g2) * g2 * P.nx / W;
    const long long n_edge = n_z + n_y;                     // no x faces: deposit_index wraps x at the source
    const unsigned blocks = (unsigned)((n_edge + 255) / 256);
    tick(c, PM_K_FOLD, 0);
    const Tiles T = tiles_of(c);
    if (P.zopen && !c->slab_packed) PM_FAIL(c, PM_EORDER, "pm_fold_ghosts (z slab): pm_slab_pack and the exchange of the slabs come first");
    const int rset = (P.zopen && c->put_step) ? 2 * c->put_parity : 0;
    const double *rlo = P.zopen ? c->slab_mem + (2 + rset) * c->slab_elems : nullptr, *rhi = P.zopen ? c->slab_mem + (3 + rset) * c->slab_elems : nullptr;
    if (c->repro) {
        if (W == 2) k_fold_ghosts<2, kReproChannels, true><<<blocks, 256, 0, c->stream>>>(P, c->buf, T, n_edge, n_z, n_y, rlo, rhi);
        else k_fold_ghosts<1, kReproChannels, true><<<blocks, 256, 0, c->stream>>>(P, c->buf, T, n_edge, n_z, n_y, rlo, rhi);
    } else {
        if (W == 2) k_fold_ghosts<2, kBufChannels, true><<<blocks, 256, 0, c->stream>>>(P, c->buf, T, n_edge, n_z, n_y, rlo, rhi);
        else k_fold_ghosts<1, kBufChannels, true><<<blocks, 256, 0, c->stream>>>(P, c->buf, T, n_edge, n_z, n_y, rlo, rhi);
    }
    int rc = check_launch(c, "k_fold_ghosts");
    tick(c, PM_K_FOLD, 1);
    if (rc != PM_OK) return rc;
    c->stage = ST_FOLDED;
    c->buffer_valid = true;
    return PM_OK;
}

template <int VEC>
static void launch_apply(pm_ctx *c, const DevState &U) {
    const DevP &P = c->P;
    const unsigned ipr = (unsigned)(P.nx / VEC);
    const unsigned n_items = (unsigned)(P.N / VEC);
    const unsigned blocks = (n_items + kApplyThreads - 1) / kApplyThreads;
    const bool tl = P.tl_num > 0.0;
#define PM_APPLY(LAM_, TL_, REPRO_, lamptr)                                                                                   \
    k_apply_limited<VEC, LAM_, TL_, REPRO_><<<blocks, kApplyThreads, 0, c->stream>>>(P, U, c->buf, tiles_of(c), c->ret, c->ret_tr, lamptr, \
                                                                                     c->repro_M, n_items, ipr)
    if (c->lam) {
        if (c->repro) { if (tl) PM_APPLY(true, true, true, c->lam); else PM_APPLY(true, false, true, c->lam); }
        else { if (tl) PM_APPLY(true, true, false, c->lam); else PM_APPLY(true, false, false, c->lam); }
    } else {
        if (c->repro) { if (tl) PM_APPLY(false, true, true, nullptr); else PM_APPLY(false, false, true, nullptr); }
        else { if (tl) PM_APPLY(false, true, false, nullptr); else PM_APPLY(false, false, false, nullptr); }
    }
#undef PM_APPLY
}

extern "C" int pm_apply_limited(pm_ctx *c, pm_state *st) {
    if (!c) return PM_EINVAL;
    if (c->stage != ST_FOLDED) PM_FAIL(c, PM_EORDER, "pm_apply_limited must follow pm_fold_ghosts");
    if (!state_ok(st)) PM_FAIL(c, PM_EINVAL, "pm_apply_limited: null state pointer");
    PM_CUDA(c, cudaSetDevice(c->device));
    const DevState U = { st->rho, st->mx, st->my, st->mz, st->etot, st->eint };
    const bool vec2 = (c->P.nx % 2 == 0) && aligned16(st->rho) && aligned16(st->mx) && aligned16(st->my) &&
                      aligned16(st->mz) && aligned16(st->etot) && aligned16(st->eint);
    tick(c, PM_K_APPLY, 0);
    if (vec2) launch_apply<2>(c, U); else launch_apply<1>(c, U);
    int rc = check_launch(c, "k_apply_limited");
    tick(c, PM_K_APPLY, 1);
    if (rc != PM_OK) return rc;
    c->stage = ST_APPLIED;
    return PM_OK;
}

extern "C" int pm_return_to_particles(pm_ctx *c, pm_sinks *sk) {
    if (!c) return PM_EINVAL;
    if (c->stage != ST_APPLIED) PM_FAIL(c, PM_EORDER, "pm_return_to_particles must follow pm_apply_limited");
    const long long nk = sk ? sk->n : 0;
    if (nk != c->n_sinks_dep) PM_FAIL(c, PM_EINVAL, "pm_return_to_particles: %lld sinks, but %lld were deposited", nk, c->n_sinks_dep);
    PM_CUDA(c, cudaSetDevice(c->device));
    if (nk > 0) {
        if (!(sk->x && sk->y && sk->z && sk->vx && sk->vy && sk->vz && sk->m)) PM_FAIL(c, PM_EINVAL, "pm_return_to_particles: null sink array");
        const DevSinks S = { nk, sk->x, sk->y, sk->z, sk->vx, sk->vy, sk->vz, sk->m, sk->dm, sk->dpx, sk->dpy, sk->dpz };
        const unsigned blocks = (unsigned)((nk + 3) / 4);
        const int *perm = c->bin_mem + c->n_sinks_dep + c->n_sne_dep;
        tick(c, PM_K_RETURN, 0);
        if (c->P.gs == 4 && !c->force_generic)
            k_return_sinks_g4<<<blocks, kFastSinkWarps * 32, 0, c->stream>>>(c->P, S, c->dt, c->sink_scal, c->ret, c->ret_tr, perm);
        else
            k_return_sinks<<<blocks, 128, 0, c->stream>>>(c->P, S, c->dt, c->sink_scal, c->ret, c->ret_tr, perm);
        int rc = check_launch(c, "k_return_sinks");
        if (rc != PM_OK) return rc;
        tick(c, PM_K_RETURN, 1);
    }
    c->stage = ST_IDLE;
    return PM_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// (f)4: z-slab decomposition (pm_slab.cuh)
// ---------------------------------------------------------------------------------------------------------------
extern "C" int pm_slab_describe(pm_ctx *c, pm_slab_desc *d) {
    if (!c || !d) return PM_EINVAL;
    if (!c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_slab_describe: the ctx was not created with z_slab = 1");
    std::memset(d, 0, sizeof(*d));
    const DevP &P = c->P;
    d->buf_bytes = c->slab_elems * (int64_t)sizeof(double);
    d->buf_send_lo = c->slab_mem; d->buf_send_hi = c->slab_mem + c->slab_elems;
    d->buf_recv_lo = c->slab_mem + 2 * c->slab_elems; d->buf_recv_hi = c->slab_mem + 3 * c->slab_elems;
    const long long plane = (long long)P.ny * P.nx, gp = (long long)P.g * plane;
    if (c->ret) {      // planes of the return mesh, in units of records of kRetWords doubles
        d->ret_bytes = gp * kRetWords * (int64_t)sizeof(double);
        d->ret_recv_lo = c->ret;                                          // ghost planes k in [-g, 0)
        d->ret_send_lo = c->ret + kRetWords * gp;                         // owned planes k in [0, g): the lower neighbour's high ghosts
        d->ret_send_hi = c->ret + kRetWords * (long long)P.nz * plane;    // owned planes k in [nz - g, nz): the upper neighbour's low ghosts
        d->ret_recv_hi = c->ret + kRetWords * ((long long)P.nz * plane + gp);   // ghost planes k in [nz, nz + g)
    }
    if (c->ret_tr) {
        d->rtr_bytes = gp * (int64_t)sizeof(double);
        d->rtr_recv_lo = c->ret_tr; d->rtr_send_lo = c->ret_tr + gp;
        d->rtr_send_hi = c->ret_tr + (long long)P.nz * plane; d->rtr_recv_hi = c->ret_tr + (long long)P.nz * plane + gp;
    }
    d->state_ghost_planes = P.g;
    return PM_OK;
}

extern "C" int pm_slab_pack(pm_ctx *c) {
    if (!c) return PM_EINVAL;
    if (!c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_slab_pack: the ctx was not created with z_slab = 1");
    if (c->stage != ST_DEPOSITED) PM_FAIL(c, PM_EORDER, "pm_slab_pack must follow pm_deposit");
    PM_CUDA(c, cudaSetDevice(c->device));
    const DevP &P = c->P;
    const long long n = 2ll * P.g * P.pk;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    if (c->repro) k_slab_pack<kReproChannels><<<blocks, 256, 0, c->stream>>>(P, c->buf, tiles_of(c), c->slab_mem, c->slab_mem + c->slab_elems);
    else k_slab_pack<kBufChannels><<<blocks, 256, 0, c->stream>>>(P, c->buf, tiles_of(c), c->slab_mem, c->slab_mem + c->slab_elems);
    int rc = check_launch(c, "k_slab_pack");
    if (rc != PM_OK) return rc;
    c->slab_packed = true;
    return PM_OK;
}

// ---- peer-memory form of the Step 2 exchange: pack + put in one kernel -----------------------------------------------------
static void slab_set_peers(pm_ctx *c, double *base_lower, double *base_upper) {
    for (int p = 0; p < 2; ++p) {
        c->put_lo[p] = base_lower + (3 + 2 * p) * c->slab_elems;      // my low ghost planes -> the lower neighbour's recv_hi
        c->put_hi[p] = base_upper + (2 + 2 * p) * c->slab_elems;      // my high ghost planes -> the upper neighbour's recv_lo
    }
    c->peers_set = true;
    c->put_parity = 1;                                                 // the first put toggles it to 0
}

static int slab_close_ipc(pm_ctx *c) {
    for (int k = 0; k < 2; ++k)
        if (c->ipc_base[k]) {
            if (k == 1 && c->ipc_base[1] == c->ipc_base[0]) { c->ipc_base[1] = nullptr; continue; }
            PM_CUDA(c, cudaIpcCloseMemHandle(c->ipc_base[k]));
            c->ipc_base[k] = nullptr;
        }
    return PM_OK;
}

extern "C" int pm_slab_connect_local(pm_ctx *c, pm_ctx *lower, pm_ctx *upper) {
    if (!c) return PM_EINVAL;
    if (!c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_slab_connect_local: the ctx was not created with z_slab = 1");
    if (!lower) lower = c;
    if (!upper) upper = c;
    for (pm_ctx *o : { lower, upper })
        if (!o->P.zopen || o->slab_elems != c->slab_elems)
            PM_FAIL(c, PM_EINVAL, "pm_slab_connect_local: the neighbour's slabs have another shape (nx, ny, ghost width and channel count must agree)");
    int rc = slab_close_ipc(c);
    if (rc != PM_OK) return rc;
    slab_set_peers(c, lower->slab_mem, upper->slab_mem);
    return PM_OK;
}

extern "C" int pm_slab_ipc_export(pm_ctx *c, void *handle, int64_t *slab_bytes) {
    if (!c) return PM_EINVAL;
    if (!handle) PM_FAIL(c, PM_EINVAL, "pm_slab_ipc_export: null handle buffer");
    if (!c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_slab_ipc_export: the ctx was not created with z_slab = 1");
    static_assert(sizeof(cudaIpcMemHandle_t) == PM_IPC_HANDLE_BYTES, "pm.h states the size of an IPC handle");
    PM_CUDA(c, cudaSetDevice(c->device));
    cudaIpcMemHandle_t h;
    PM_CUDA(c, cudaIpcGetMemHandle(&h, c->slab_mem));
    std::memcpy(handle, &h, sizeof(h));
    if (slab_bytes) *slab_bytes = c->slab_elems * (int64_t)sizeof(double);
    return PM_OK;
}

extern "C" int pm_slab_connect_ipc(pm_ctx *c, const void *handle_lower, const void *handle_upper) {
    if (!c) return PM_EINVAL;
    if (!c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_slab_connect_ipc: the ctx was not created with z_slab = 1");
    PM_CUDA(c, cudaSetDevice(c->device));
    int rc = slab_close_ipc(c);
    if (rc != PM_OK) return rc;
    double *base[2] = { c->slab_mem, c->slab_mem };                   // NULL handle: this ctx is its own neighbour on that side
    const void *hs[2] = { handle_lower, handle_upper };
    for (int k = 0; k < 2; ++k) {
        if (!hs[k]) continue;
        if (k == 1 && hs[0] && std::memcmp(hs[0], hs[1], PM_IPC_HANDLE_BYTES) == 0) {     // two ranks: both neighbours are the same peer
            c->ipc_base[1] = c->ipc_base[0]; base[1] = base[0];
            continue;
        }
        cudaIpcMemHandle_t h;
        std::memcpy(&h, hs[k], sizeof(h));
        void *ptr = nullptr;
        PM_CUDA(c, cudaIpcOpenMemHandle(&ptr, h, cudaIpcMemLazyEnablePeerAccess));
        c->ipc_base[k] = ptr; base[k] = static_cast<double *>(ptr);
    }
    slab_set_peers(c, base[0], base[1]);
    return PM_OK;
}

extern "C" int pm_slab_put(pm_ctx *c) {
    if (!c) return PM_EINVAL;
    if (!c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_slab_put: the ctx was not created with z_slab = 1");
    if (!c->peers_set) PM_FAIL(c, PM_EORDER, "pm_slab_put: connect the neighbours first (pm_slab_connect_ipc / pm_slab_connect_local)");
    if (c->stage != ST_DEPOSITED || c->slab_packed) PM_FAIL(c, PM_EORDER, "pm_slab_put must follow pm_deposit (once)");
    PM_CUDA(c, cudaSetDevice(c->device));
    const DevP &P = c->P;
    const long long n = 2ll * P.g * P.pk;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    c->put_parity ^= 1;
    double *lo = c->put_lo[c->put_parity], *hi = c->put_hi[c->put_parity];
    if (c->repro) k_slab_pack<kReproChannels><<<blocks, 256, 0, c->stream>>>(P, c->buf, tiles_of(c), lo, hi);
    else k_slab_pack<kBufChannels><<<blocks, 256, 0, c->stream>>>(P, c->buf, tiles_of(c), lo, hi);
    int rc = check_launch(c, "k_slab_pack (put)");
    if (rc != PM_OK) return rc;
    c->slab_packed = true;
    c->put_step = true;
    return PM_OK;
}

extern "C" int pm_create_sinks(pm_ctx *c, pm_state *st, int64_t max_new, double *x, double *y, double *z, double *vx,
                               double *vy, double *vz, double *m, int64_t *n_new) {
    if (!c) return PM_EINVAL;
    if (!n_new) PM_FAIL(c, PM_EINVAL, "pm_create_sinks: n_new is NULL");
    *n_new = 0;
    if (!state_ok(st)) PM_FAIL(c, PM_EINVAL, "pm_create_sinks: null state pointer");
    if (c->P.gs == 0 || !(c->P.tl_num > 0.0)) PM_FAIL(c, PM_EINVAL, "pm_create_sinks needs rk_sink > 0 and truelove_J > 0");
    if (c->stage == ST_DEPOSITED || c->stage == ST_FOLDED) PM_FAIL(c, PM_EORDER, "pm_create_sinks: finish the step (pm_apply_limited) first");
    if (max_new < 0 || max_new >= (1ll << 31) || (max_new > 0 && !(x && y && z && vx && vy && vz && m))) PM_FAIL(c, PM_EINVAL, "pm_create_sinks: bad output arrays");
    PM_CUDA(c, cudaSetDevice(c->device));
    const DevP &P = c->P;
    const int cap = (int)max_new;
    const int nblocks = (int)((P.N + 255) / 256), nscan = (nblocks + kScanChunk - 1) / kScanChunk;
    // scratch (ints): total | block counts [nblocks] | chunk sums [nscan] | list [cap]; then the flags (bytes, one per cell)
    const long long need = 1 + (long long)nblocks + nscan + cap + (P.N + 3) / 4;
    if (need > c->create_cap) {
        if (c->create_mem) { PM_CUDA(c, cudaFree(c->create_mem)); c->create_mem = nullptr; c->create_cap = 0; }
        PM_CUDA(c, cudaMalloc(&c->create_mem, (size_t)need * sizeof(int)));
        c->create_cap = need;
    }
    int *total = c->create_mem, *bcount = total + 1, *sums = bcount + nblocks, *list = sums + nscan;
    unsigned char *flag = reinterpret_cast<unsigned char *>(list + cap);
    const DevState U = { st->rho, st->mx, st->my, st->mz, st->etot, st->eint };
    int rc;
    PM_CUDA(c, cudaMemsetAsync(total, 0, (size_t)(1 + nblocks) * sizeof(int), c->stream));
    // (iii) needs the folded accretion channel of the last deposit; before the first deposit there is none and the test is skipped
    if (c->ever_deposited && !c->buffer_valid) PM_FAIL(c, PM_EORDER, "pm_create_sinks: the retained buffer is not folded (call pm_fold_ghosts)");
    k_create_find<<<nblocks, 256, 0, c->stream>>>(P, U, c->buffer_valid ? c->buf : nullptr, tiles_of(c), flag, bcount);
    if ((rc = check_launch(c, "k_create_find")) != PM_OK) return rc;
    k_bin_scan_local<<<nscan, 256, 0, c->stream>>>(bcount, nblocks, sums);
    if ((rc = check_launch(c, "k_bin_scan_local")) != PM_OK) return rc;
    k_bin_scan_sums<<<1, 1024, 0, c->stream>>>(sums, nscan);
    if ((rc = check_launch(c, "k_bin_scan_sums")) != PM_OK) return rc;
    k_create_compact<<<nblocks, 256, 0, c->stream>>>(P.N, flag, bcount, sums, kScanChunk, list, cap, total);
    if ((rc = check_launch(c, "k_create_compact")) != PM_OK) return rc;
    PM_CUDA(c, cudaMemcpyAsync(c->err_host + 1, total, sizeof(int), cudaMemcpyDeviceToHost, c->stream));   // the only host traffic
    PM_CUDA(c, cudaStreamSynchronize(c->stream));
    const int found = c->err_host[1];
    if (found > 0 && found <= cap) {
        k_create_apply<<<(unsigned)((found + 127) / 128), 128, 0, c->stream>>>(P, U, list, found, x, y, z, vx, vy, vz, m);
        if ((rc = check_launch(c, "k_create_apply")) != PM_OK) return rc;
        PM_CUDA(c, cudaStreamSynchronize(c->stream));
    }
    *n_new = found;
    return PM_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// (f)3: PM gravity (L95, L107): Steps 1, 2, 5 with the cloud-in-cell kernel, interpolation + kick, drift
// ---------------------------------------------------------------------------------------------------------------
// Gravity works in buffer channel 1 (the first supernova channel): it is free between steps, its reset here is a plain
// sweep of that one channel, and the tile flags are not involved -- the next pm_deposit rewrites them anyway.  Channel 0
// (the retained accretion buffer of L108 / L177) and its flags are left alone, so pm_create_sinks still works afterwards.
static int fold_gravity_channel(pm_ctx *c, double *gbuf) {
    const DevP &P = c->P;
    const long long g2 = 2 * P.g;
    const int W = P.nx % 2 == 0 ? 2 : 1;
    const long long n_z = g2 * P.ny * P.nx / W;
    const long long n_y = (long long)(P.nz - g2) * g2 * P.nx / W;
    const long long n_edge = n_z + n_y;
    const unsigned blocks = (unsigned)((n_edge + 255) / 256);
    if (W == 2) k_fold_ghosts<2, 1, false><<<blocks, 256, 0, c->stream>>>(P, gbuf, tiles_of(c), n_edge, n_z, n_y, nullptr, nullptr);
    else k_fold_ghosts<1, 1, false><<<blocks, 256, 0, c->stream>>>(P, gbuf, tiles_of(c), n_edge, n_z, n_y, nullptr, nullptr);
    return check_launch(c, "k_fold_ghosts<1 channel>");
}

// Particles in a1 bin order for the gravity kernels (a counting sort by host tile, no comparison sort): *perm_out lists the
// particle indices tile by tile, or is NULL for small sets (order does not matter below the L2 size).  The permutation only
// decides which thread takes which particle; results do not depend on it (interpolation) or only through the order of the
// atomic additions (deposit).
constexpr long long kGravSortMin = 1 << 16;
static int grav_order(pm_ctx *c, const double *x, const double *y, const double *z, long long n, const int **perm_out) {
    *perm_out = nullptr;
    if (n < kGravSortMin) return PM_OK;
    if (n >= (1ll << 31)) PM_FAIL(c, PM_EINVAL, "too many particles");
    const DevP &P = c->P;
    const int nkeys = 2 * P.ntile + 1;
    const int nscan = (nkeys + kScanChunk - 1) / kScanChunk;
    if (c->gperm_valid && c->gperm_x == x && c->gperm_n == n) { *perm_out = c->grav_mem + n; return PM_OK; }
    c->gperm_valid = false;
    const long long need = 2 * n + nkeys + nscan + nkeys;
    if (need > c->grav_cap) {
        if (c->grav_mem) { PM_CUDA(c, cudaFree(c->grav_mem)); c->grav_mem = nullptr; c->grav_cap = 0; }
        const long long cap = need + need / 4;
        cudaError_t e = cudaMalloc(&c->grav_mem, (size_t)cap * sizeof(int));
        if (e != cudaSuccess) { c->grav_mem = nullptr; PM_FAIL(c, PM_ENOMEM, "cudaMalloc of bins failed: %s", cudaGetErrorString(e)); }
        c->grav_cap = cap;
    }
    int *keys = c->grav_mem, *perm = keys + n, *counts = perm + n, *sums = counts + nkeys, *fillc = sums + nscan;
    int rc;
    PM_CUDA(c, cudaMemsetAsync(counts, 0, (size_t)(nkeys + nscan + nkeys) * sizeof(int), c->stream));
    const unsigned blocks = (unsigned)((n + 255) / 256);
    k_bin_count<<<blocks, 256, 0, c->stream>>>(P, x, y, z, n, nullptr, nullptr, nullptr, 0, keys, counts, nullptr);
    if ((rc = check_launch(c, "k_bin_count")) != PM_OK) return rc;
    k_bin_scan_local<<<nscan, 256, 0, c->stream>>>(counts, nkeys, sums);
    if ((rc = check_launch(c, "k_bin_scan_local")) != PM_OK) return rc;
    k_bin_scan_sums<<<1, 1024, 0, c->stream>>>(sums, nscan);
    if ((rc = check_launch(c, "k_bin_scan_sums")) != PM_OK) return rc;
    k_bin_fill<<<blocks, 256, 0, c->stream>>>(keys, counts, fillc, sums, perm, n, n);
    if ((rc = check_launch(c, "k_bin_fill")) != PM_OK) return rc;
    c->gperm_x = x; c->gperm_n = n; c->gperm_valid = true;
    *perm_out = perm;
    return PM_OK;
}

extern "C" int pm_gravity_deposit(pm_ctx *c, const double *rho_gas, int64_t n, const double *x, const double *y, const double *z,
                                  const double *m, double *rho_tot) {
    if (!c) return PM_EINVAL;
    if (n < 0 || !rho_tot) PM_FAIL(c, PM_EINVAL, "pm_gravity_deposit: null output or negative particle count");
    if (n > 0 && !(x && y && z && m)) PM_FAIL(c, PM_EINVAL, "pm_gravity_deposit: null particle array");
    if (c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_gravity_deposit: not available on a z slab (the gravity calls are single-domain)");
    if (c->stage == ST_DEPOSITED || c->stage == ST_FOLDED)
        PM_FAIL(c, PM_EORDER, "pm_gravity_deposit: the buffer mesh is in use (finish the exchange step first)");
    PM_CUDA(c, cudaSetDevice(c->device));
    const DevP &P = c->P;
    double *const gbuf = c->buf + P.Nb;      // channel 1; see fold_gravity_channel
    c->grav_in_ch1 = true;
    int rc;
    PM_CUDA(c, cudaMemsetAsync(gbuf, 0, (size_t)P.Nb * sizeof(double), c->stream));     // Step 1: "initialized to zero" (L59)
    if (n > 0) {
        const int *perm;
        if ((rc = grav_order(c, x, y, z, n, &perm)) != PM_OK) return rc;
        k_grav_deposit<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(P, x, y, z, m, n, perm, gbuf, c->err_flag);
        if ((rc = check_launch(c, "k_grav_deposit")) != PM_OK) return rc;
    }
    if ((rc = fold_gravity_channel(c, gbuf)) != PM_OK) return rc;                           // Step 2
    const bool vec = P.nx % 2 == 0 && aligned16(rho_tot) && (!rho_gas || aligned16(rho_gas));
    const long long work = vec ? P.N / 2 : P.N;
    long long blocks = (work + 255) / 256;
    const long long cap = (long long)c->sm_count * 32;
    if (blocks > cap) blocks = cap;
    if (vec) k_grav_apply<2><<<(unsigned)blocks, 256, 0, c->stream>>>(P, rho_gas, gbuf, rho_tot);   // Step 5
    else k_grav_apply<1><<<(unsigned)blocks, 256, 0, c->stream>>>(P, rho_gas, gbuf, rho_tot);
    return check_launch(c, "k_grav_apply");
}

extern "C" int pm_gravity_kick(pm_ctx *c, const double *gx, const double *gy, const double *gz, int64_t n, const double *x,
                               const double *y, const double *z, double *vx, double *vy, double *vz, double dt, double *ax,
                               double *ay, double *az) {
    if (!c) return PM_EINVAL;
    if (n < 0 || !(gx && gy && gz)) PM_FAIL(c, PM_EINVAL, "pm_gravity_kick: null acceleration mesh or negative particle count");
    if (n == 0) return PM_OK;
    if (!(x && y && z)) PM_FAIL(c, PM_EINVAL, "pm_gravity_kick: null position array");
    const bool has_v = vx || vy || vz, has_a = ax || ay || az;
    if (has_v && !(vx && vy && vz)) PM_FAIL(c, PM_EINVAL, "pm_gravity_kick: give all of vx, vy, vz or none");
    if (has_a && !(ax && ay && az)) PM_FAIL(c, PM_EINVAL, "pm_gravity_kick: give all of ax, ay, az or none");
    if (!has_v && !has_a) PM_FAIL(c, PM_EINVAL, "pm_gravity_kick: nothing to write (no velocities, no acceleration output)");
    if (c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_gravity_kick: not available on a z slab (the gravity calls are single-domain)");
    PM_CUDA(c, cudaSetDevice(c->device));
    const int *perm;
    int rc;
    if ((rc = grav_order(c, x, y, z, n, &perm)) != PM_OK) return rc;
    k_grav_kick<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->P, gx, gy, gz, n, x, y, z, vx, vy, vz, dt, ax, ay, az, perm, c->err_flag);
    return check_launch(c, "k_grav_kick");
}

extern "C" int pm_drift(pm_ctx *c, int64_t n, double *x, double *y, double *z, const double *vx, const double *vy, const double *vz,
                        double dt) {
    if (!c) return PM_EINVAL;
    if (n < 0) PM_FAIL(c, PM_EINVAL, "pm_drift: negative particle count");
    if (n == 0) return PM_OK;
    if (!(x && y && z && vx && vy && vz)) PM_FAIL(c, PM_EINVAL, "pm_drift: null particle array");
    if (c->stage == ST_APPLIED)
        PM_FAIL(c, PM_EORDER, "pm_drift: pm_return_to_particles needs the positions of the preceding pm_deposit; call it first");
    PM_CUDA(c, cudaSetDevice(c->device));
    c->gperm_valid = false;      // positions change: the cached order is stale (still a valid permutation, but not reused)
    k_drift<<<(unsigned)((n + 255) / 256), 256, 0, c->stream>>>(c->P, n, x, y, z, vx, vy, vz, dt, c->err_flag);
    return check_launch(c, "k_drift");
}

extern "C" int pm_check(pm_ctx *c) {
    if (!c) return PM_EINVAL;
    PM_CUDA(c, cudaSetDevice(c->device));
    PM_CUDA(c, cudaMemcpyAsync(c->err_host, c->err_flag, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    PM_CUDA(c, cudaStreamSynchronize(c->stream));
    if (*c->err_host & 1) {
        PM_CUDA(c, cudaMemsetAsync(c->err_flag, 0, sizeof(int), c->stream));
        PM_FAIL(c, PM_EDOMAIN, "a particle lies outside the domain [x0, x0 + n dx)");
    }
    return PM_OK;
}

// One step with HOST buffers, in two halves.  begin: enqueue the upload of the inputs (up_stream), the four calls (the ctx's
// stream, after the upload) and the download of the results (down_stream, after the kernels); end: wait for the download.
// Two slots with staging of their own: the caller may begin slot 1 - s while slot s is still downloading, and PCIe carries
// both directions at once.  The kernels of the two slots run one after the other on the ctx's stream (there is one buffer mesh).
extern "C" int pm_step_host_begin(pm_ctx *c, int slot_id, pm_state *hs, pm_sinks *hk, const pm_sne *hn, double dt) {
    if (!c) return PM_EINVAL;
    if (slot_id < 0 || slot_id > 1) PM_FAIL(c, PM_EINVAL, "pm_step_host_begin: slot must be 0 or 1");
    if (!state_ok(hs)) PM_FAIL(c, PM_EINVAL, "pm_step_host: null state pointer");
    if (c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_step_host: not available on a z slab (the exchanges between the calls are the caller's)");
    pm_ctx::HostSlot &S = c->slot[slot_id];
    if (S.busy) PM_FAIL(c, PM_EORDER, "pm_step_host_begin: slot %d is in flight (pm_step_host_end first)", slot_id);
    PM_CUDA(c, cudaSetDevice(c->device));
    const long long N = c->P.N, nk = hk ? hk->n : 0, nn = hn ? hn->n : 0;
    int rc;
    if ((rc = grow(c, &S.stg_state, &S.stg_state_cap, 6 * N)) != PM_OK) return rc;
    if ((rc = grow(c, &S.stg_sinks, &S.stg_sinks_cap, 11 * nk)) != PM_OK) return rc;
    if ((rc = grow(c, &S.stg_sne, &S.stg_sne_cap, 8 * nn)) != PM_OK) return rc;
    if (!c->up_stream) {
        PM_CUDA(c, cudaStreamCreateWithFlags(&c->up_stream, cudaStreamNonBlocking));
        PM_CUDA(c, cudaStreamCreateWithFlags(&c->down_stream, cudaStreamNonBlocking));
        for (int k = 0; k < 2; ++k) {
            PM_CUDA(c, cudaEventCreateWithFlags(&c->slot[k].ev_up, cudaEventDisableTiming));
            PM_CUDA(c, cudaEventCreateWithFlags(&c->slot[k].ev_done, cudaEventDisableTiming));
            PM_CUDA(c, cudaEventCreateWithFlags(&c->slot[k].ev_down, cudaEventDisableTiming));
        }
    }
    cudaStream_t s = c->stream, up = c->up_stream, down = c->down_stream;
    double *hst[6] = { hs->rho, hs->mx, hs->my, hs->mz, hs->etot, hs->eint };
    // the slot's staging was last read by its own download, which pm_step_host_end has waited for
    for (int f = 0; f < 6; ++f) PM_CUDA(c, cudaMemcpyAsync(S.stg_state + f * N, hst[f], N * 8, cudaMemcpyHostToDevice, up));
    pm_state ds = { S.stg_state, S.stg_state + N, S.stg_state + 2 * N, S.stg_state + 3 * N, S.stg_state + 4 * N, S.stg_state + 5 * N };
    pm_sinks dk; std::memset(&dk, 0, sizeof(dk));
    pm_sne dn; std::memset(&dn, 0, sizeof(dn));
    if (nk > 0) {
        const double *src[7] = { hk->x, hk->y, hk->z, hk->vx, hk->vy, hk->vz, hk->m };
        for (int f = 0; f < 7; ++f) {
            if (!src[f]) PM_FAIL(c, PM_EINVAL, "pm_step_host: null sink array");
            PM_CUDA(c, cudaMemcpyAsync(S.stg_sinks + f * nk, src[f], nk * 8, cudaMemcpyHostToDevice, up));
        }
        double *b = S.stg_sinks;
        dk.n = nk; dk.x = b; dk.y = b + nk; dk.z = b + 2 * nk; dk.vx = b + 3 * nk; dk.vy = b + 4 * nk; dk.vz = b + 5 * nk; dk.m = b + 6 * nk;
        dk.dm = b + 7 * nk; dk.dpx = b + 8 * nk; dk.dpy = b + 9 * nk; dk.dpz = b + 10 * nk;
    }
    if (nn > 0) {
        const double *src[8] = { hn->x, hn->y, hn->z, hn->vx, hn->vy, hn->vz, hn->e_sn, hn->m_ej };
        for (int f = 0; f < 8; ++f) {
            if (!src[f]) PM_FAIL(c, PM_EINVAL, "pm_step_host: null SN array");
            PM_CUDA(c, cudaMemcpyAsync(S.stg_sne + f * nn, src[f], nn * 8, cudaMemcpyHostToDevice, up));
        }
        double *b = S.stg_sne;
        dn.n = nn; dn.x = b; dn.y = b + nn; dn.z = b + 2 * nn; dn.vx = b + 3 * nn; dn.vy = b + 4 * nn; dn.vz = b + 5 * nn;
        dn.e_sn = b + 6 * nn; dn.m_ej = b + 7 * nn;
    }
    PM_CUDA(c, cudaEventRecord(S.ev_up, up));
    PM_CUDA(c, cudaStreamWaitEvent(s, S.ev_up, 0));
    if ((rc = pm_deposit(c, &ds, nk > 0 ? &dk : nullptr, nn > 0 ? &dn : nullptr, dt)) != PM_OK) return rc;
    if ((rc = pm_fold_ghosts(c)) != PM_OK) return rc;
    if ((rc = pm_apply_limited(c, &ds)) != PM_OK) return rc;
    if ((rc = pm_return_to_particles(c, nk > 0 ? &dk : nullptr)) != PM_OK) return rc;
    PM_CUDA(c, cudaEventRecord(S.ev_done, s));
    PM_CUDA(c, cudaStreamWaitEvent(down, S.ev_done, 0));
    for (int f = 0; f < 6; ++f) PM_CUDA(c, cudaMemcpyAsync(hst[f], S.stg_state + f * N, N * 8, cudaMemcpyDeviceToHost, down));
    if (nk > 0) {
        double *dst[8] = { hk->vx, hk->vy, hk->vz, hk->m, hk->dm, hk->dpx, hk->dpy, hk->dpz };
        for (int f = 0; f < 8; ++f)
            if (dst[f]) PM_CUDA(c, cudaMemcpyAsync(dst[f], S.stg_sinks + (3 + f) * nk, nk * 8, cudaMemcpyDeviceToHost, down));
    }
    PM_CUDA(c, cudaMemcpyAsync(c->err_host, c->err_flag, sizeof(int), cudaMemcpyDeviceToHost, down));
    PM_CUDA(c, cudaEventRecord(S.ev_down, down));
    S.busy = true;
    return PM_OK;
}

extern "C" int pm_step_host_end(pm_ctx *c, int slot_id) {
    if (!c) return PM_EINVAL;
    if (slot_id < 0 || slot_id > 1) PM_FAIL(c, PM_EINVAL, "pm_step_host_end: slot must be 0 or 1");
    pm_ctx::HostSlot &S = c->slot[slot_id];
    if (!S.busy) PM_FAIL(c, PM_EORDER, "pm_step_host_end: slot %d has no step in flight", slot_id);
    PM_CUDA(c, cudaSetDevice(c->device));
    S.busy = false;
    PM_CUDA(c, cudaEventSynchronize(S.ev_down));
    if (*c->err_host & 1) {
        PM_CUDA(c, cudaMemsetAsync(c->err_flag, 0, sizeof(int), c->stream));
        PM_FAIL(c, PM_EDOMAIN, "a particle lies outside the domain [x0, x0 + n dx)");
    }
    return PM_OK;
}

extern "C" int pm_step_host(pm_ctx *c, pm_state *hs, pm_sinks *hk, const pm_sne *hn, double dt) {
    int rc = pm_step_host_begin(c, 0, hs, hk, hn, dt);
    if (rc != PM_OK) return rc;
    return pm_step_host_end(c, 0);
}

// ---- pm_step_graph ---------------------------------------------------------------------------------------------
// One step = twelve launches and a memset; on small meshes (BASELINE configs 1-3) the host's launch calls take longer than the
// kernels run.  The four calls are therefore captured once into a CUDA graph and replayed while the argument pointers, the
// particle counts and dt stay what they were: first call with a set of arguments -> plain calls (they put the scratch memory in
// place: no allocation may happen under capture); second call -> the same calls under stream capture, instantiate, launch; from
// the third on -> one cudaGraphLaunch.  The kernels read positions, masses and the state from memory, so a run whose particles
// move and whose gas evolves replays the same graph.
static int step_calls(pm_ctx *c, pm_state *st, pm_sinks *sk, const pm_sne *sn, double dt) {
    int rc = pm_deposit(c, st, sk, sn, dt);
    if (rc == PM_OK) rc = pm_fold_ghosts(c);
    if (rc == PM_OK) rc = pm_apply_limited(c, st);
    if (rc == PM_OK && sk && sk->n > 0) rc = pm_return_to_particles(c, sk);
    return rc;
}

// The graph is captured from, and replayed on, a stream of the ctx's own (the caller's may be a default stream, which cannot be
// captured); two events order it after what the caller's stream holds and the caller's stream after it.
static int graph_launch(pm_ctx *c) {
    PM_CUDA(c, cudaEventRecord(c->gev_in, c->stream));
    PM_CUDA(c, cudaStreamWaitEvent(c->gstream, c->gev_in, 0));
    PM_CUDA(c, cudaGraphLaunch(c->gexec, c->gstream));
    PM_CUDA(c, cudaEventRecord(c->gev_out, c->gstream));
    PM_CUDA(c, cudaStreamWaitEvent(c->stream, c->gev_out, 0));
    return PM_OK;
}

extern "C" int pm_step_graph(pm_ctx *c, pm_state *st, pm_sinks *sk, const pm_sne *sn, double dt) {
    if (!c) return PM_EINVAL;
    if (!state_ok(st)) PM_FAIL(c, PM_EINVAL, "pm_step_graph: null state pointer");
    if (c->P.zopen) PM_FAIL(c, PM_EINVAL, "pm_step_graph: not available on a z slab (the exchange sits between the calls)");
    pm_ctx::GraphKey key;
    std::memset(&key, 0, sizeof(key));
    key.st = *st; key.dt = dt;
    if (sk) key.sk = *sk;
    if (sn) key.sn = *sn;
    const bool capturable = !c->timing;      // the events of PM_FLAG_TIMING must not end up inside a graph
    const bool same = c->gstate > 0 && std::memcmp(&key, &c->gkey, sizeof(key)) == 0;
    if (capturable && same && c->gstate == 2) {
        PM_CUDA(c, cudaSetDevice(c->device));
        const int rc = graph_launch(c);
        if (rc != PM_OK) return rc;
        // what the four calls leave behind on the host side
        c->launches += c->glaunches;
        c->n_sinks_dep = sk ? sk->n : 0; c->n_sne_dep = sn ? sn->n : 0; c->dt = dt;
        c->ever_deposited = true; c->grav_in_ch1 = false; c->buffer_valid = true;
        c->stage = (sk && sk->n > 0) ? ST_IDLE : ST_APPLIED;
        return PM_OK;
    }
    if (capturable && same && c->gstate == 1) {
        PM_CUDA(c, cudaSetDevice(c->device));
        if (!c->gstream) {
            PM_CUDA(c, cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking));
            PM_CUDA(c, cudaEventCreateWithFlags(&c->gev_in, cudaEventDisableTiming));
            PM_CUDA(c, cudaEventCreateWithFlags(&c->gev_out, cudaEventDisableTiming));
        }
        const long long l0 = c->launches;
        cudaStream_t const user = c->stream;
        cudaGraph_t graph = nullptr;
        cudaError_t e = cudaStreamBeginCapture(c->gstream, cudaStreamCaptureModeThreadLocal);
        if (e == cudaSuccess) {
            c->stream = c->gstream;                          // every launch of the four calls goes to c->stream
            const int rc = step_calls(c, st, sk, sn, dt);
            c->stream = user;
            e = cudaStreamEndCapture(c->gstream, &graph);
            if (rc == PM_OK && e == cudaSuccess && graph) {
                if (c->gexec) { cudaGraphExecDestroy(c->gexec); c->gexec = nullptr; }
                e = cudaGraphInstantiate(&c->gexec, graph, 0);
                cudaGraphDestroy(graph);
                if (e == cudaSuccess) {
                    c->glaunches = c->launches - l0;
                    c->gstate = 2;
                    return graph_launch(c);
                }
            } else if (graph) cudaGraphDestroy(graph);
        }
        cudaGetLastError();                    // capture refused or broken: forget it and do the step the plain way
        c->launches = l0;
        c->gstate = 0;
        c->stage = ST_IDLE;
    }
    const int rc = step_calls(c, st, sk, sn, dt);
    if (rc == PM_OK && capturable) { c->gkey = key; c->gstate = 1; }
    else c->gstate = 0;
    return rc;
}

extern "C" int pm_debug_graph_state(pm_ctx *c, int32_t *state) {
    if (!c || !state) return PM_EINVAL;
    *state = c->gstate;
    return PM_OK;
}

// ---- test-only views ---------------------------------------------------------------------------------------------
static int materialize_tiles(pm_ctx *c) {
    PM_CUDA(c, cudaSetDevice(c->device));
    k_tiles_materialize<<<(unsigned)((c->ntiles + 3) / 4), 128, 0, c->stream>>>(c->P, c->buf, tiles_of(c), c->repro, c->grav_in_ch1, (int)c->ntiles);
    return check_launch(c, "k_tiles_materialize");
}

extern "C" int pm_debug_buffer(pm_ctx *c, int channel, const double **dev_ptr, int64_t dims[3], int64_t *origin, int32_t *ghost) {
    if (!c || !dev_ptr || channel < 0 || channel >= kBufChannels) return PM_EINVAL;
    {   // the raw mesh is only readable once the zeros that stale tiles stand for have been stored (test-only, not timed)
        int rc = materialize_tiles(c);
        if (rc != PM_OK) return rc;
    }
    *dev_ptr = c->buf + (long long)channel * c->P.Nb;
    if (dims) { dims[0] = c->P.nz + 2 * c->P.g; dims[1] = c->P.ny + 2 * c->P.g; dims[2] = c->P.pj; }
    if (origin) *origin = (long long)c->P.g * c->P.pk + (long long)c->P.g * c->P.pj + c->P.gx;
    if (ghost) *ghost = c->P.g;
    return PM_OK;
}

extern "C" int pm_debug_tile_counts(pm_ctx *c, int64_t *n_tiles, int64_t *live_k, int64_t *live_n) {
    if (!c || !n_tiles || !live_k || !live_n) return PM_EINVAL;
    PM_CUDA(c, cudaSetDevice(c->device));
    unsigned char *h = new (std::nothrow) unsigned char[(size_t)c->ntiles];
    if (!h) return PM_ENOMEM;
    cudaError_t e = cudaMemcpyAsync(h, c->tile_live, (size_t)c->ntiles, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { delete[] h; snprintf(c->msg, sizeof(c->msg), "pm_debug_tile_counts: %s", cudaGetErrorString(e)); return PM_ECUDA; }
    int64_t k = 0, n = 0;
    for (long long t = 0; t < c->ntiles; ++t) { k += (h[t] & kLiveK) ? 1 : 0; n += (h[t] & kLiveN) ? 1 : 0; }
    delete[] h;
    *n_tiles = c->ntiles; *live_k = k; *live_n = n;
    return PM_OK;
}

extern "C" int pm_debug_return_mesh(pm_ctx *c, int word, const double **dev_ptr) {
    if (!c || !dev_ptr || word < 0 || word >= kRetWords || !c->ret) return PM_EINVAL;
    *dev_ptr = c->ret + (long long)kRetWords * c->P.zoff + word;   // record of OWNED cell q at 4 q (behind the ghost planes of a slab)
    return PM_OK;
}

extern "C" int pm_debug_round_buffers(pm_ctx *c) {
    if (!c) return PM_EINVAL;
    if (!c->repro) PM_FAIL(c, PM_EINVAL, "pm_debug_round_buffers needs PM_FLAG_REPRODUCIBLE");
    if (!c->buffer_valid) PM_FAIL(c, PM_EORDER, "pm_debug_round_buffers: fold first");
    int rc0 = materialize_tiles(c);
    if (rc0 != PM_OK) return rc0;
    const DevP &P = c->P;
    if (P.nx % 2 == 0) k_repro_round<2><<<(unsigned)((P.N / 2 + 255) / 256), 256, 0, c->stream>>>(P, c->buf, c->repro_M, P.N / 2);
    else k_repro_round<1><<<(unsigned)((P.N + 255) / 256), 256, 0, c->stream>>>(P, c->buf, c->repro_M, P.N);
    return check_launch(c, "k_repro_round");
}

extern "C" int pm_debug_lambda(pm_ctx *c, const double **dev_ptr) {
    if (!c || !dev_ptr || !c->lam) return PM_EINVAL;
    *dev_ptr = c->lam;
    return PM_OK;
}

extern "C" int pm_debug_sink_scalars(pm_ctx *c, const double **dev_ptr, int64_t *n) {
    if (!c || !dev_ptr || !n || !(c->prm.flags & PM_FLAG_DEBUG_SCALARS)) return PM_EINVAL;
    *dev_ptr = c->dbg_sink; *n = c->n_sinks_dep;
    return PM_OK;
}

extern "C" int pm_debug_sn_scalars(pm_ctx *c, const double **dev_ptr, int64_t *n) {
    if (!c || !dev_ptr || !n || !(c->prm.flags & PM_FLAG_DEBUG_SCALARS)) return PM_EINVAL;
    *dev_ptr = c->dbg_sn; *n = c->n_sne_dep;
    return PM_OK;
}

extern "C" int pm_debug_stencil(pm_ctx *c, int kind, double x, double y, double z, int32_t *dev_counts, int32_t *host_ijk, int32_t *side) {
    if (!c || !dev_counts || !host_ijk || !side || kind < 0 || kind > 1) return PM_EINVAL;
    const int g = kind == 0 ? c->P.gs : c->P.gn;
    if (g == 0) PM_FAIL(c, PM_EINVAL, "pm_debug_stencil: that particle kind is unused");
    PM_CUDA(c, cudaSetDevice(c->device));
    int *d_ijk = nullptr;
    PM_CUDA(c, cudaMalloc(&d_ijk, 3 * sizeof(int)));
    const size_t smem = kind == 1 ? sn_table_bytes(2 * g + 1, c->P.nsub) : 0;
    k_debug_stencil<<<1, 32, smem, c->stream>>>(c->P, kind, x, y, z, dev_counts, d_ijk);
    int rc = check_launch(c, "k_debug_stencil");
    if (rc == PM_OK) {
        cudaError_t e = cudaMemcpyAsync(host_ijk, d_ijk, 3 * sizeof(int), cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) { snprintf(c->msg, sizeof(c->msg), "pm_debug_stencil: %s", cudaGetErrorString(e)); rc = PM_ECUDA; }
    }
    cudaFree(d_ijk);
    *side = 2 * g + 1;
    return rc;
}

// ---- measurement helpers ---------------------------------------------------------------------------------------------
extern "C" int pm_kernel_times(pm_ctx *c, float *ms, int32_t n) {
    if (!c || !ms || n < PM_NUM_KERNELS) return PM_EINVAL;
    if (!c->timing) PM_FAIL(c, PM_EINVAL, "pm_kernel_times needs PM_FLAG_TIMING");
    PM_CUDA(c, cudaSetDevice(c->device));
    PM_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < PM_NUM_KERNELS; ++k) {
        ms[k] = 0.0f;
        if (c->ev_used[k]) PM_CUDA(c, cudaEventElapsedTime(&ms[k], c->ev[k][0], c->ev[k][1]));
    }
    return PM_OK;
}

// fp64 RED throughput for the deposit's pattern: rows of 7 consecutive doubles (4 rows + 4 idle lanes per warp
// instruction), the same row position in `channels` planes, pseudo-random row positions over the footprint.
__device__ __forceinline__ unsigned probe_hash(unsigned x) {
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
}

__global__ void __launch_bounds__(256) k_probe_red(double *__restrict__ buf, unsigned long long plane, int channels, int iters) {
    const unsigned tid = blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned warp = tid >> 5, lane = tid & 31;
    const unsigned row = lane / 7, col = lane - row * 7;
    if (row >= 4) return;
    const unsigned long long nrow = plane / 8;
    for (int it = 0; it < iters; ++it) {
        const unsigned long long r = probe_hash((warp * 4 + row) * 977u + it * 0x9e3779b9u) % nrow;
        double *p = buf + r * 8 + col + (probe_hash(warp + it) & 1);
        for (int f = 0; f < channels; ++f) atomicAdd(p + f * plane, 1.0);
    }
}

extern "C" int pm_probe_red_f64(pm_ctx *c, int64_t footprint_bytes, int32_t channels, double *gops) {
    if (!c || !gops || channels < 1 || channels > 8 || footprint_bytes < (int64_t)channels * 4096) return PM_EINVAL;
    PM_CUDA(c, cudaSetDevice(c->device));
    const unsigned long long plane = ((unsigned long long)footprint_bytes / 8 / channels) & ~7ull;
    double *buf = nullptr;
    cudaError_t e = cudaMalloc(&buf, (plane * channels + 16) * sizeof(double));
    if (e != cudaSuccess) { cudaGetLastError(); PM_FAIL(c, PM_ENOMEM, "pm_probe_red_f64: cudaMalloc failed: %s", cudaGetErrorString(e)); }
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    const int blocks = c->sm_count * 16, iters = 64;
    cudaMemsetAsync(buf, 0, (plane * channels + 16) * sizeof(double), c->stream);
    k_probe_red<<<blocks, 256, 0, c->stream>>>(buf, plane, channels, iters);        // warm-up
    cudaEventRecord(a, c->stream);
    k_probe_red<<<blocks, 256, 0, c->stream>>>(buf, plane, channels, iters);
    cudaEventRecord(b, c->stream);
    e = cudaStreamSynchronize(c->stream);
    float ms = 0.0f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(buf);
    if (e != cudaSuccess) { snprintf(c->msg, sizeof(c->msg), "pm_probe_red_f64: %s", cudaGetErrorString(e)); return PM_ECUDA; }
    const double ops = (double)blocks * 8 * 28 * iters * channels;      // 8 warps per CTA, 28 active lanes
    *gops = ops / (ms * 1e-3) / 1e9;
    return PM_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// pm_gravity_deposit_noalloc: the PM-gravity mass deposit (Steps 1, 2, 5; L51, L95) for callers that cannot allocate --
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  Same kernels and the same
// arithmetic as pm_gravity_deposit; the ghost-zoned accumulation mesh (the scratch of Step 1, L59) lives in a file-scope
// __device__ array instead of a ctx's buffer mesh, so no ctx and no allocation is needed.  Every GPU that loads the library
// holds the array until the process exits (PM_NOALLOC_SCRATCH_BYTES).
//
// In host code the name g_noalloc_scratch is a host-side stand-in, not a device address: the address the kernels get comes
// from cudaGetSymbolAddress, asked once per device with that device current (noalloc_scratch below).
//
// Layout: [0, 32) doubles = 256 bytes of flag words ([0] as int: "a particle lies outside the domain"); then the mesh,
// (nx + 4)(ny + 2)(nz + 2) doubles (one ghost layer, r_K = dx for cloud-in-cell, R40; x origin rounded to even as in a ctx).
// All calls share the array and it keeps the last call's contents: every call clears the part it uses first.  Two calls
// whose work overlaps on the GPU (different streams, different host threads) race on it.
// ---------------------------------------------------------------------------------------------------------------
constexpr long long kNoallocFlagDoubles = 32;
constexpr long long kNoallocMeshMax = PM_NOALLOC_MAX_GHOSTED_CELLS;
static_assert((kNoallocFlagDoubles + kNoallocMeshMax) * sizeof(double) == PM_NOALLOC_SCRATCH_BYTES, "pm.h states the size of the array");
static __device__ __align__(256) double g_noalloc_scratch[kNoallocFlagDoubles + kNoallocMeshMax];

constexpr int kNoallocMaxDevices = 64;
static std::mutex g_noalloc_mu;
static double *g_noalloc_ptr[kNoallocMaxDevices];       // device address of g_noalloc_scratch, per device; NULL = not asked yet
static thread_local char g_noalloc_msg[384] = "";

#define NOALLOC_FAIL(code, ...) do { snprintf(g_noalloc_msg, sizeof(g_noalloc_msg), __VA_ARGS__); return (code); } while (0)
#define NOALLOC_CUDA(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { \
    snprintf(g_noalloc_msg, sizeof(g_noalloc_msg), "%s failed: %s", #call, cudaGetErrorString(e_)); return PM_ECUDA; } } while (0)

// Set-up, once per device: makes `device` current and asks the runtime where this device keeps g_noalloc_scratch.
static int noalloc_scratch(int device, double **out) {
    if (device < 0 || device >= kNoallocMaxDevices) NOALLOC_FAIL(PM_EINVAL, "device %d: the no-alloc entry point serves devices 0..%d", device, kNoallocMaxDevices - 1);
    NOALLOC_CUDA(cudaSetDevice(device));
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[device]) {
        double *p = nullptr;
        NOALLOC_CUDA(cudaGetSymbolAddress((void **)&p, g_noalloc_scratch));
        if (!p) NOALLOC_FAIL(PM_ECUDA, "cudaGetSymbolAddress gave a null address for the scratch array on device %d", device);
        g_noalloc_ptr[device] = p;
    }
    *out = g_noalloc_ptr[device];
    return PM_OK;
}

extern "C" const char *pm_noalloc_last_error(void) { return g_noalloc_msg; }

extern "C" int pm_noalloc_setup(int device) {
    double *p;
    return noalloc_scratch(device, &p);
}

extern "C" int pm_gravity_deposit_noalloc(int device, void *cuda_stream, int32_t nx, int32_t ny, int32_t nz, const double *x0,
                                          double dx, const double *rho_gas, int64_t n, const double *x, const double *y,
                                          const double *z, const double *m, double *rho_tot, int32_t *outside) {
    g_noalloc_msg[0] = 0;
    if (!x0 || !rho_tot || n < 0 || n >= (1ll << 31)) NOALLOC_FAIL(PM_EINVAL, "pm_gravity_deposit_noalloc: null x0 / rho_tot, or a particle count outside [0, 2^31)");
    if (n > 0 && !(x && y && z && m)) NOALLOC_FAIL(PM_EINVAL, "pm_gravity_deposit_noalloc: null particle array");
    if (nx < 3 || ny < 3 || nz < 3 || !(dx > 0.0)) NOALLOC_FAIL(PM_EINVAL, "pm_gravity_deposit_noalloc: needs dx > 0 and at least 3 cells per axis (R32 with one ghost layer)");
    const long long Nb = ((long long)nx + 4) * ((long long)ny + 2) * ((long long)nz + 2);
    if (Nb > kNoallocMeshMax)
        NOALLOC_FAIL(PM_EINVAL, "pm_gravity_deposit_noalloc: a mesh of %d x %d x %d cells needs (nx + 4)(ny + 2)(nz + 2) = %lld doubles of scratch; "
                     "the static array holds PM_NOALLOC_MAX_GHOSTED_CELLS = %lld (cubes up to 66^3 fit); use pm_gravity_deposit on a ctx",
                     (int)nx, (int)ny, (int)nz, Nb, kNoallocMeshMax);
    double *scr;
    int rc;
    if ((rc = noalloc_scratch(device, &scr)) != PM_OK) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;

    DevP P;
    std::memset(&P, 0, sizeof(P));
    P.nx = nx; P.ny = ny; P.nz = nz;
    P.g = 1; P.gx = 2;
    P.pj = nx + 2 * P.gx; P.pk = P.pj * (ny + 2 * P.g);
    P.N = (long long)nx * ny * nz; P.Nb = Nb;
    P.dx = dx; P.inv_dx = 1.0 / dx; P.V = dx * dx * dx;
    for (int a = 0; a < 3; ++a) P.x0[a] = x0[a];

    int *const flag = reinterpret_cast<int *>(scr);
    double *const mesh = scr + kNoallocFlagDoubles;
    // Step 1: "all cells initialized to zero" (L59) -- and the flag words: the array still holds the previous call's sums
    NOALLOC_CUDA(cudaMemsetAsync(scr, 0, (size_t)(kNoallocFlagDoubles + Nb) * sizeof(double), stream));
    if (n > 0) {
        k_grav_deposit<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(P, x, y, z, m, n, nullptr, mesh, flag);
        NOALLOC_CUDA(cudaGetLastError());
    }
    {                                                                                     // Step 2 (Eq. 3), one channel, W = 1 (g odd)
        const long long g2 = 2 * P.g;
        const long long n_z = g2 * P.ny * P.nx;
        const long long n_y = (long long)(P.nz - g2) * g2 * P.nx;
        const long long n_edge = n_z + n_y;
        k_fold_ghosts<1, 1, false><<<(unsigned)((n_edge + 255) / 256), 256, 0, stream>>>(P, mesh, Tiles{nullptr, nullptr}, n_edge, n_z, n_y, nullptr, nullptr);
        NOALLOC_CUDA(cudaGetLastError());
    }
    const bool vec = P.nx % 2 == 0 && aligned16(rho_tot) && (!rho_gas || aligned16(rho_gas));      // Step 5 (Eq. 6, eta = 1)
    const long long work = vec ? P.N / 2 : P.N;
    const unsigned blocks = (unsigned)((work + 255) / 256);          // at most 1024 CTAs at the maximum mesh
    if (vec) k_grav_apply<2><<<blocks, 256, 0, stream>>>(P, rho_gas, mesh, rho_tot);
    else k_grav_apply<1><<<blocks, 256, 0, stream>>>(P, rho_gas, mesh, rho_tot);
    NOALLOC_CUDA(cudaGetLastError());
    if (outside) NOALLOC_CUDA(cudaMemcpyAsync(outside, flag, sizeof(int), cudaMemcpyDeviceToDevice, stream));
    return PM_OK;
}
