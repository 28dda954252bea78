/*
 * pm.h -- C ABI of libpm_b200: one particle-mesh-particle exchange step on one B200 (sm_100a).
 *
 * Method: arxiv 2509.18261 (He et al.), /root/reference/PAPER.md.  "L" numbers are PAPER.md lines,
 * "R" numbers are the readings listed in DESIGN.md.
 *
 *   pm_deposit             Step 1, Eq. 2 (L59-65) with the sink recipe of Sec. 3.1.1 (Eqs. 7-11, 13; L117-159)
 *                          and the supernova recipe of Sec. 3.2.1 (Eqs. 17-20; L203-230): every particle adds its
 *                          deposition function dU^s_ijk into a ghost-zoned buffer mesh with fp64 atomic additions.
 *   pm_fold_ghosts         Step 2, Eq. 3 (L67-71): ghost-zone contents are added to the owning real zones.  On one
 *                          GPU the "other rank" is the periodic image, so this is an in-device periodic fold.  (y and z ghost
 *                          zones; along x, the fastest axis, particles add to the periodic image directly.)
 *   pm_apply_limited       Steps 3 + 5, Eqs. 4 and 6 (L73-77, L89-93) fused: the cell-wise limiters (Eqs. 15-16,
 *                          L161-171, with BASELINE's max-removable-fraction and density floor; Eq. 21) and
 *                          U := U + eta dU^sum, in place on the caller's conserved state.
 *   pm_return_to_particles Step 4, Eq. 5 (L79-87): u_s := u_s - sum_ijk eta_ijk dU^s_ijk V_ijk for every sink
 *                          (supernova particles skip this step, L201).
 *   pm_gravity_deposit / pm_gravity_kick / pm_drift   PM gravity for the particles' own motion (L95, L107): Steps 1, 2, 5
 *                          with the cloud-in-cell kernel, interpolation back with the same kernel, kick-drift-kick.
 *   z_slab = 1, pm_slab_pack / pm_slab_put   Step 2 across ranks (L97): a domain cut along z; the z ghost planes travel to the
 *                          two neighbours as messages, or are stored straight into their receive slabs by the pack kernel.
 *   pm_gravity_deposit_noalloc   the gravity deposit without a ctx and without any allocation (static device scratch).
 *
 * All pointers inside pm_state / pm_sinks / pm_sne are DEVICE pointers (cudaMalloc'ed by the caller, e.g. torch
 * allocations) unless a function says "host".  Every array is fp64, contiguous.  Mesh fields hold nx*ny*nz values,
 * x fastest ((k*ny + j)*nx + i), no ghost zones, periodic in all three directions.  The library never frees or
 * reallocates caller memory.  The ctx owns: the ghost-zoned buffer mesh (6 channels), the return mesh (eta and the
 * pre-step cell velocity, 4 words per cell, written where a sink removed mass), per-particle scratch.
 *
 * Execution: every call enqueues kernels on the ctx's CUDA stream and returns without synchronising the host
 * (except pm_step_host, pm_check and pm_destroy).  Within a step the calls must come in the order
 * deposit -> fold -> apply -> return (return may be skipped when there are no sinks); otherwise PM_EORDER.
 * The buffer mesh stays valid (as dU^sum, L108) until the next pm_deposit, which resets it.
 *
 * Buffer reset ("all cells initialized to zero", L59): the mesh is cut into tiles of 8^3 cells with a liveness flag.  pm_deposit
 * marks and zeroes the tiles this step's particles can add into (known from the particle bins); all other tiles are stale, and
 * fold, apply and sink creation take them as zeros without reading them.
 *
 * Which call is allowed when (PM_EORDER otherwise).  "in step" = after pm_deposit, before pm_apply_limited has returned:
 *   pm_deposit              any time (abandons an unfinished step)
 *   pm_fold_ghosts          directly after pm_deposit          pm_apply_limited        directly after pm_fold_ghosts
 *   pm_return_to_particles  directly after pm_apply_limited (may be skipped when there are no sinks)
 *   pm_create_sinks         not in step; after a step it needs the folded buffer of that step
 *   pm_gravity_deposit      not in step (it works in buffer channel 1; the retained accretion channel 0 is left alone)
 *   pm_gravity_kick         any time (own scratch memory; reads no buffer)
 *   pm_drift                not between pm_apply_limited and pm_return_to_particles (Step 4 needs the deposit's positions)
 *
 * Errors: every function returns 0 on success or a negative pm_status; no exceptions, no aborts, no output.
 * pm_last_error(ctx) gives a human-readable message for the last failure on that ctx.
 */
#ifndef PM_B200_H
#define PM_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    PM_OK = 0,
    PM_EINVAL = -1,   /* null / misaligned pointer, bad parameter, grid smaller than 2g+1 cells, particle count changed */
    PM_ENOMEM = -2,   /* device allocation failed */
    PM_ECUDA = -3,    /* a CUDA call or kernel failed (sticky); text in pm_last_error */
    PM_EORDER = -4,   /* call sequence violated */
    PM_EDOMAIN = -5   /* a particle lies outside [x0, x0 + n dx); detected on device, reported by pm_check / pm_step_host */
} pm_status;

/* supernova regime selector, Eq. 19 (L223) */
enum { PM_SN_AUTO = 0, PM_SN_FORCE_EJ = 1, PM_SN_FORCE_ST = 2, PM_SN_FORCE_MC = 3 };

/* Plain data, copied at pm_create.  Units are the caller's; nothing is assumed about them. */
typedef struct {
    int32_t nx, ny, nz;          /* owned cells per axis (periodic); each must be >= 2g+1, g = ghost width */
    int32_t sn_nsub;             /* omega sub-samples per axis, 1..8 (R17); 1 = binary centre test */
    int32_t sn_regime;           /* PM_SN_* */
    int32_t flags;               /* PM_FLAG_* */
    double dx;                   /* cell size; V_ijk = dx^3 (uniform mesh, R33) */
    double x0[3];                /* lower corner of cell (0,0,0) */
    double G, gamma;             /* gravitational constant; adiabatic index for c_s^2 = gamma (gamma-1) e_int/rho */
    double cs_iso;               /* > 0: use this constant sound speed instead (R6) */
    double rk_sink, rk_sn;       /* kernel radii r_K in length units (L117, L201); 0 = that particle kind is unused */
    double bondi_lambda;         /* lambda of Eq. 8; e^{3/2}/4 in the paper (L130) */
    double f_max_remove;         /* largest fraction of a cell's mass sinks may remove per step (L161: 0.25) */
    double rho_floor;            /* accretion never takes a cell below this density */
    double sn_eps_k, sn_rm_ej, sn_rm_mc;     /* 0.28, 0.027, 1 (L223-225) */
    double sn_msf_coeff, sn_msf_exp;         /* M_sf = coeff (n_H / nh_unit)^exp (L203) */
    double sn_psnr_coeff, sn_psnr_exp;       /* P_snr = coeff (n_H / nh_unit)^exp, Eq. 20 (L229) */
    double sn_mu_h, sn_nh_unit;              /* mass per H nucleus; unit of n_H */
    double sn_eint_theta;        /* Eq. 21 floor: e_min = theta rho_2 (e_int,1/rho_1); 1 = as printed, 0 = e_int >= 0 only (R25) */
    double truelove_J;           /* Jeans number J of Eq. 12, rho_Tr = J^2 pi c_s^2 / (G dx^2); 0.25 in the paper (L148); 0 = the Truelove
                                  * terms of Eqs. 13-14 and 16 are off (all BASELINE configs) */
    int32_t z_slab;              /* 0: one periodic domain (Step 2 is the in-device fold).  1: this ctx holds the nz planes of one z slab
                                  * of a larger domain (periodic in x and y inside the ctx, cut along z): see pm_slab_describe */
    int32_t pad_;
} pm_params;

enum {
    PM_FLAG_DEBUG_SCALARS = 1,   /* keep per-particle scalars (pm_debug_sink_scalars / pm_debug_sn_scalars) */
    PM_FLAG_DEBUG_LAMBDA = 2,    /* keep the Eq. 21 lambda of every cell (pm_debug_lambda) */
    PM_FLAG_GENERIC_KERNELS = 4, /* always use the generic (any radius, any n_sub) deposit / return kernels */
    PM_FLAG_TIMING = 8,          /* bracket every kernel with CUDA events on the ctx's stream (pm_kernel_times) */
    PM_FLAG_SMEM_TILES = 32,     /* supernova bins (8^3 tiles) with >= 48 particles are accumulated by one CTA in a shared-memory tile
                                  * accumulator (14^3 cells x 5 channels) and added to the buffer mesh once, instead of one fp64 RED per
                                  * cell and particle.  Same results up to the order of the additions.  Off by default: on B200 the
                                  * direct path is faster at every density measured; ignored in Appendix A mode */
    PM_FLAG_REPRODUCIBLE = 16    /* Appendix A (L586-615): three more buffer channels (two error scales, contribution counts); the apply
                                  * pass rounds the folded sums as it reads them: the step no longer depends on the order of
                                  * the atomic additions, except with probability ~2^-M per cell */
};

typedef struct { double *rho, *mx, *my, *mz, *etot, *eint; } pm_state;

/* Sink particles, u_s = (m, m v) (L49).  x,y,z are never modified.  dm, dpx, dpy, dpz are optional outputs
 * (may be NULL): the mass and momentum actually returned to each sink in this step (Eq. 5). */
typedef struct {
    int64_t n;
    const double *x, *y, *z;
    double *vx, *vy, *vz, *m;
    double *dm, *dpx, *dpy, *dpz;
} pm_sinks;

/* Supernova particles exploding in this step (never modified, L201). */
typedef struct {
    int64_t n;
    const double *x, *y, *z, *vx, *vy, *vz, *e_sn, *m_ej;
} pm_sne;

typedef struct pm_ctx pm_ctx;

/* Create a context on CUDA device `device`, launching on `cuda_stream` (a cudaStream_t; NULL = default stream).
 * Allocates the buffer mesh ((n+2g)^3 x 6 channels) and, if rk_sink > 0, the return mesh (4 n^3 words). */
int pm_create(const pm_params *params, int device, void *cuda_stream, pm_ctx **out);

/* Step 1.  Resets the buffer mesh, then deposits every sink and SN (reading the PRE-step state).  sinks / sne may be
 * NULL or have n == 0.  dt is the time step of Eq. 13.  Caches per-sink scalars (mdot, r_acc, sum w) for Step 4. */
int pm_deposit(pm_ctx *ctx, const pm_state *state, const pm_sinks *sinks, const pm_sne *sne, double dt);

/* Step 2.  Adds every ghost cell's contents to the periodically wrapped owned cell, in a fixed image order (the sum
 * order of a cell is the same in every run, cf. Appendix A).  Ghost cells keep their values. */
int pm_fold_ghosts(pm_ctx *ctx);

/* Steps 3 + 5.  In place on the caller's state.  Leaves eta and the pre-step velocity for Step 4. */
int pm_apply_limited(pm_ctx *ctx, pm_state *state);

/* Step 4.  Must be given the same sinks (same n, same positions) as the preceding pm_deposit. */
int pm_return_to_particles(pm_ctx *ctx, pm_sinks *sinks);

/* ---- z-slab decomposition.  Step 2 as the paper states it: "add the contents of the ghost zones on each
 * rank to the corresponding real zones on other ranks" (L67-71, Eq. 3), the one non-local step (L97).  A ctx created with
 * z_slab = 1 owns the planes k in [0, nz) of its slab; rank r's lower neighbour is r - 1, its upper neighbour r + 1 (periodic
 * in the rank index).  What changes for the caller:
 *   * every mesh array in pm_state holds (nz + 2g) ny nx values: g ghost planes (g = state_ghost_planes), the nz owned planes,
 *     g ghost planes; the ghost planes must hold the neighbours' boundary planes BEFORE pm_deposit (the halo exchange every
 *     hydro code already has; particles near a z face read gas across it).  pm_apply_limited updates owned planes only.
 *   * sequence:  pm_deposit -> pm_slab_pack -> [send buf_send_lo to the lower neighbour's buf_recv_hi, buf_send_hi to the upper
 *     neighbour's buf_recv_lo] -> pm_fold_ghosts -> pm_apply_limited -> [send ret_send_lo to the lower neighbour's ret_recv_hi,
 *     ret_send_hi to the upper neighbour's ret_recv_lo; the same for rtr_* when truelove_J > 0] -> pm_return_to_particles.
 *     The transfers are the caller's (NCCL / torch.distributed / cudaMemcpyPeer); they must be ordered after the preceding and
 *     before the following call on the ctx's stream.  The second exchange is the owner -> ghost copy of (eta, v_old) that
 *     Step 4 needs for sinks whose kernel crosses a z face (L79); the paper does not mention it (R16).
 *   * a slab message is [channel][g planes][ny + 2g][row pitch] doubles, unfolded; the receiver adds the images of a cell in
 *     the same fixed order as the single-domain fold (Appendix A), so one rank that is its own neighbour reproduces
 *     the periodic fold bit for bit.
 * Not available on a slab: pm_step_host and the PM-gravity calls. */
typedef struct {
    void *buf_send_lo, *buf_send_hi, *buf_recv_lo, *buf_recv_hi;   /* DEVICE, ctx-owned, buf_bytes each */
    int64_t buf_bytes;
    void *ret_send_lo, *ret_send_hi, *ret_recv_lo, *ret_recv_hi;   /* DEVICE, inside the ctx's return mesh, ret_bytes each (NULL / 0: no sinks) */
    int64_t ret_bytes;
    void *rtr_send_lo, *rtr_send_hi, *rtr_recv_lo, *rtr_recv_hi;   /* the same for the Truelove excess kept for Step 4 (NULL / 0 when off) */
    int64_t rtr_bytes;
    int32_t state_ghost_planes;                                     /* g */
    int32_t pad_;
} pm_slab_desc;
int pm_slab_describe(pm_ctx *ctx, pm_slab_desc *out);
/* After pm_deposit: fill buf_send_lo / buf_send_hi from the buffer mesh's z ghost planes (stale tiles as zeros). */
int pm_slab_pack(pm_ctx *ctx);

/* Peer-memory form of the Step 2 exchange: compute step and transfer in ONE kernel.  pm_slab_put replaces "pm_slab_pack, then
 * send / receive": the pack kernel stores this rank's low z ghost planes straight into the LOWER neighbour's receive slab and
 * its high ones into the UPPER neighbour's, through peer-mapped device memory (NVLink / NVSwitch between GPUs of a node; plain
 * device memory when both ranks share a GPU or a rank is its own neighbour).  No staging copy, no library collective.
 *   set-up, once:  every rank calls pm_slab_ipc_export (a 64-byte CUDA IPC handle of its slab memory), the handles travel by any
 *                  host channel (torch.distributed.all_gather_object in sharded.py), and every rank calls pm_slab_connect_ipc with
 *                  its two neighbours' handles (NULL = this ctx is its own neighbour on that side; with two ranks both handles are
 *                  the same peer's and it is opened once).  Neighbours that live in the SAME process (several ctxs, one process)
 *                  are connected with pm_slab_connect_local instead (CUDA IPC handles cannot be opened by their own process).
 *   every step:    pm_deposit -> pm_slab_put -> [all ranks: synchronise the ctx's stream, then a host barrier: every put has
 *                  landed] -> pm_fold_ghosts -> ... as above.
 * The receive slabs exist twice and pm_slab_put alternates between the two sets, so a put of step n + 1 never lands in memory
 * the neighbour's fold of step n may still be reading, and ONE barrier per step suffices: a rank leaves the barrier of step n + 1
 * only after its stream, and with it its fold of step n, has drained.  All ranks must call pm_slab_put in every step of a run
 * (the sets alternate in lock step); pm_slab_pack steps (which use set 0) may not be mixed in between.
 * The neighbours' slab memory must stay alive while this ctx can still put: destroy the ctxs of a run together, after a barrier.
 * Errors: PM_EORDER (not connected; not directly after pm_deposit), PM_EINVAL (not a slab ctx; neighbour of another shape),
 * PM_ECUDA (IPC: the peer's GPU is not peer-accessible from this one). */
#define PM_IPC_HANDLE_BYTES 64
int pm_slab_ipc_export(pm_ctx *ctx, void *handle /* HOST, PM_IPC_HANDLE_BYTES */, int64_t *slab_bytes /* HOST, optional: bytes of one slab */);
int pm_slab_connect_ipc(pm_ctx *ctx, const void *handle_lower, const void *handle_upper);
int pm_slab_connect_local(pm_ctx *ctx, pm_ctx *lower, pm_ctx *upper);      /* NULL = ctx itself */
int pm_slab_put(pm_ctx *ctx);

/* Margin M of Appendix A (N_bit = log2 r + 52 + M; default 28, the paper's example, L612).  Needs PM_FLAG_REPRODUCIBLE. */
int pm_set_repro_margin(pm_ctx *ctx, int32_t M);

/* Sink particle creation (Sec. 3.1.2); needs rk_sink > 0 and truelove_J > 0.  Call between steps (after
 * pm_apply_limited / pm_return_to_particles, before the next pm_deposit).  A cell creates a sink if rho > rho_Tr (Eq. 12),
 * it is a strict local density maximum among the cells whose centres lie within rk_sink of its own (periodic), and the
 * accretion channel of the retained buffer mesh is zero there (no sink's kernel covers it, L177; before the first deposit
 * this test is skipped; after a pm_deposit that was not folded: PM_EORDER).  New sink: cell centre, m = (rho - rho_Tr) V, velocity of the cell; the cell is left at rho_Tr
 * with the same velocity and specific energies (L183).  state: DEVICE, modified in place.  x .. m: DEVICE arrays of
 * max_new doubles, filled in increasing cell-index order (an ordered compaction on the device; only the count goes to
 * the host).  *n_new (HOST) = number of cells found; if it exceeds max_new NOTHING is created and the state is unchanged
 * (call again with larger arrays).  Synchronises. */
int pm_create_sinks(pm_ctx *ctx, pm_state *state, int64_t max_new, double *x, double *y, double *z, double *vx, double *vy,
                    double *vz, double *m, int64_t *n_new);

/* ---- PM gravity: Steps 1, 2 and 5 only (L95: "no limiting ... interactions do not modify particle
 * properties, only mesh properties"; L107: sinks and star particles move under "a standard PM gravity method, which we
 * implement using steps 1, 2, and 5", kick-drift-kick).  The Poisson solve between pm_gravity_deposit and pm_gravity_kick is
 * the host code's (multigrid, L427) and is not part of this library: the acceleration mesh is an input.
 * Kernel W: cloud-in-cell (R40).  Per axis s = (x - x0)/dx - 1/2, i0 = floor(s), f = s - i0; cells i0, i0 + 1 get 1 - f, f;
 * W_ijk = (W_z W_y) W_x; r_K = dx, so one ghost layer contains it (L59).  All pointers DEVICE, fp64, contiguous; particle
 * arrays hold n values, mesh arrays nx*ny*nz (x fastest, no ghosts).  Particles must lie in [x0, x0 + n dx) (else
 * PM_EDOMAIN at the next pm_check).  Asynchronous on the ctx's stream.
 * Order of work: from 65536 particles on, both kernels take the particles in the a1 bin order (a counting sort of the
 * host tiles on the device, no comparison sort; the particle arrays themselves are never permuted), which keeps the mesh
 * sectors of neighbouring particles together in DRAM pages and L2.  The order is cached in the ctx (in scratch memory of its
 * own) between a pm_gravity_deposit and the pm_gravity_kick on the same x pointer and n, and dropped by pm_drift.  Results
 * do not depend on it except through the order of the deposit's atomic additions. */

/* rho_tot := rho_gas + sum_s m_s W(x_ijk - x_s) / V (L51: "depositing particle mass into the gas density field for the
 * purposes of computing the gravitational potential").  Step 1: buffer channel 0 is zeroed and receives the eight fp64
 * atomic additions of every particle, ghost layer included; Step 2: pm_fold_ghosts on that channel; Step 5: the sum is
 * written to rho_tot (eta = 1).  rho_gas may be NULL (particles only) and may alias rho_tot.  n may be 0.  Uses channel 1 of the
 * ctx's buffer mesh (free between steps; swept to zero here): not allowed between pm_deposit and pm_apply_limited (PM_EORDER).
 * The retained accretion channel of L108 / L177 (channel 0) is not touched, so pm_create_sinks still works afterwards. */
int pm_gravity_deposit(pm_ctx *ctx, const double *rho_gas, int64_t n, const double *x, const double *y, const double *z,
                       const double *m, double *rho_tot);

/* Mesh -> particle interpolation with the same W (L27), fused with a kick (L107): a_s = sum_ijk W(x_ijk - x_s) g_ijk over
 * the particle's eight cells (periodic; summed in the order k, j, i, low cell first), then v_s += a_s dt (dt = half the
 * step for each of the two kicks).  gx, gy, gz: acceleration meshes.  vx, vy, vz: all NULL = interpolate only.  ax, ay, az:
 * optional outputs of a_s, all NULL = not stored.  At least one of the two groups must be given. */
int pm_gravity_kick(pm_ctx *ctx, const double *gx, const double *gy, const double *gz, int64_t n, const double *x,
                    const double *y, const double *z, double *vx, double *vy, double *vz, double dt, double *ax, double *ay,
                    double *az);

/* Drift: x_s += v_s dt, brought back into the periodic box by whole box lengths (R41: a result that rounds onto the upper
 * face is put on the lower face).  Positions are modified in place -- the one call that moves particles; not allowed
 * between pm_apply_limited and pm_return_to_particles (PM_EORDER).  A non-finite result, or one more than 1e6 box lengths
 * away, raises PM_EDOMAIN at the next pm_check and is stored unwrapped. */
int pm_drift(pm_ctx *ctx, int64_t n, double *x, double *y, double *z, const double *vx, const double *vy, const double *vz,
             double dt);

/* ---- one entry point that allocates nothing -------------------------------------------------------------------
 * pm_gravity_deposit for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid it): no ctx, no cudaMalloc / cudaFree / allocating library routine, on any call.  The ghost-zoned accumulation
 * mesh of Step 1 (L59) lives in ONE file-scope __device__ array of PM_NOALLOC_SCRATCH_BYTES (2.5 MiB + 256 bytes) that every
 * GPU loading the library holds until the process exits.  Limit: (nx + 4)(ny + 2)(nz + 2) <= PM_NOALLOC_MAX_GHOSTED_CELLS
 * (cubes up to 66^3 cells fit; one ghost layer, the x origin rounded up to 2 cells); a larger mesh is refused with PM_EINVAL and a message
 * that names the limit -- use a ctx for it.  At least 3 cells per axis (R32).
 *
 * Same operation, kernels and argument meaning as pm_gravity_deposit: rho_tot := rho_gas + sum_s m_s W(x_ijk - x_s) / V (L51,
 * cloud-in-cell, R40), rho_gas may be NULL and may alias rho_tot, all array pointers DEVICE fp64 (particle arrays n values,
 * meshes nx*ny*nz, x fastest), x0 = HOST pointer to the 3 coordinates of the low corner.  Particles are taken in the order
 * given (no bin ordering: the mesh fits in L2).  outside: optional DEVICE int32; receives 1 when some particle lay outside
 * [x0, x0 + n dx) (it was skipped), else 0 -- the PM_EDOMAIN of pm_check, without a synchronisation.
 * Asynchronous on cuda_stream (a cudaStream_t, NULL = the legacy default stream) of `device`; the caller owns every buffer.
 *
 * The scratch array is shared by all calls on a device and keeps the last call's contents; every call clears the part it uses
 * first (stream-ordered).  Calls whose GPU work can overlap -- different streams, different host threads -- RACE on it:
 * serialise them (one stream, or events).  The first call on a device looks the array's device address up
 * (cudaGetSymbolAddress, once per device); pm_noalloc_setup(device) does only that, for callers that want it out of the way
 * before a capture starts.  Errors: PM_EINVAL (arguments, mesh too large), PM_ECUDA; pm_noalloc_last_error() returns the
 * message of the calling thread's last failing call ("" after a success). */
#define PM_NOALLOC_MAX_GHOSTED_CELLS 327680
#define PM_NOALLOC_SCRATCH_BYTES ((PM_NOALLOC_MAX_GHOSTED_CELLS + 32) * 8)
int pm_noalloc_setup(int device);
int pm_gravity_deposit_noalloc(int device, void *cuda_stream, int32_t nx, int32_t ny, int32_t nz, const double *x0, double dx,
                               const double *rho_gas, int64_t n, const double *x, const double *y, const double *z,
                               const double *m, double *rho_tot, int32_t *outside);
const char *pm_noalloc_last_error(void);

/* Synchronise the ctx's stream and report PM_ECUDA / PM_EDOMAIN raised by earlier asynchronous work. */
int pm_check(pm_ctx *ctx);

/* One whole step with DEVICE buffers as ONE call: pm_deposit, pm_fold_ghosts, pm_apply_limited and (when there are sinks)
 * pm_return_to_particles, replayed from a CUDA graph.  A step is twelve kernel launches and a memset; on small meshes the
 * host's launch calls take longer than the kernels run.  The first call with a given set of arguments (all pointers in state,
 * sinks and sne, the particle counts, dt) makes the plain calls; the second captures the same calls from the ctx's stream into
 * a graph and launches it; from the third on the call is one cudaGraphLaunch.  The kernels read particle data and state from
 * memory, so moving particles and evolving gas replay the same graph; any change of a pointer, a count or dt starts over with
 * plain calls.  Same results as the four calls (same kernels, same order).  The graph runs on a stream of the ctx's own, ordered
 * after the work already in the ctx's stream and before what is enqueued there next (two events per call), so the ctx's stream
 * may be a default stream.  With PM_FLAG_TIMING the plain calls are made every time.  Not on a z slab (PM_EINVAL).
 * Asynchronous; errors as for the four calls. */
int pm_step_graph(pm_ctx *ctx, pm_state *state, pm_sinks *sinks, const pm_sne *sne, double dt);

/* One whole step with HOST buffers (the end-to-end path): copies state and particles host -> device into
 * ctx-owned staging (allocated on first use), runs deposit, fold, apply, return, copies the state and the sink
 * fields (vx, vy, vz, m and the optional dm, dp*) back, and synchronises.  All pointers in the three structs are
 * HOST pointers here (pinned memory recommended). */
int pm_step_host(pm_ctx *ctx, pm_state *host_state, pm_sinks *host_sinks, const pm_sne *host_sne, double dt);

/* The same in two halves, for callers that have the NEXT step's inputs ready in other host buffers (a host code that double
 * buffers its mesh): pm_step_host_begin enqueues upload, the four calls and download of one step in slot 0 or 1 and returns
 * without waiting; pm_step_host_end waits for that slot's results (and reports PM_EDOMAIN / PM_ECUDA).  Each slot has device
 * staging of its own, uploads and downloads use two more streams, so the upload of one slot runs while the other slot still
 * downloads (PCIe carries both directions at once); the kernels of the two slots run one after the other.  The host buffers
 * of a slot must stay untouched between begin and end.  pm_step_host = begin + end on slot 0. */
int pm_step_host_begin(pm_ctx *ctx, int slot, pm_state *host_state, pm_sinks *host_sinks, const pm_sne *host_sne, double dt);
int pm_step_host_end(pm_ctx *ctx, int slot);

int pm_destroy(pm_ctx *ctx);

const char *pm_last_error(const pm_ctx *ctx);

/* Number of kernels this ctx has launched so far (bench.py's gpu_launches). */
int64_t pm_launch_count(const pm_ctx *ctx);

/* Device time of each kernel group in the most recent step, in milliseconds, measured with CUDA events recorded on the
 * ctx's stream around the launches (needs PM_FLAG_TIMING; synchronises).  ms (HOST, n >= PM_NUM_KERNELS floats):
 * PM_K_BIN (the four binning kernels), PM_K_ZERO (tile stamping + reset), PM_K_SINKS, PM_K_SNE, PM_K_FOLD, PM_K_APPLY,
 * PM_K_RETURN; a group that did not run reports 0. */
enum { PM_K_BIN = 0, PM_K_ZERO = 1, PM_K_SINKS = 2, PM_K_SNE = 3, PM_K_FOLD = 4, PM_K_APPLY = 5, PM_K_RETURN = 6, PM_NUM_KERNELS = 7 };
int pm_kernel_times(pm_ctx *ctx, float *ms, int32_t n);

/* Measured fp64 RED (atomic add without return) throughput of this device for the deposit's access pattern: every
 * warp adds to rows of 7 consecutive doubles at pseudo-random row positions in `channels` planes spread over
 * `footprint_bytes` of ctx-allocated scratch (freed before returning).  *gops (HOST) receives 1e9 lane-additions per
 * second.  footprint below the 126 MB L2 measures the L2 atomic units, far above it the HBM-miss path.  Synchronises. */
int pm_probe_red_f64(pm_ctx *ctx, int64_t footprint_bytes, int32_t channels, double *gops);

/* ---- test-only views (not timed) ---------------------------------------------------------------------------- */

/* Buffer channel 0 = accretion d rho^sum (signed, <= 0, R1); 1..5 = SN d rho, d px, d py, d pz, d E.
 * The channel is a contiguous (dims[0], dims[1], dims[2]) = (nz+2g, ny+2g, row pitch) array, x fastest; the row pitch
 * is nx + 2*gx with gx = g rounded up to even (keeps 128-bit accesses aligned).  *origin = element offset of owned
 * cell (0,0,0); owned cell (i,j,k) sits at origin + (k*dims[1] + j)*dims[2] + i, ghost cells at i,j,k in [-g, n+g).
 * *ghost = g.  Stale tiles (no particle touched them in this step) are filled with the zeros they stand for first.
 * The x ghost columns (i < 0, i >= nx) exist for alignment only and stay empty: particles wrap x where they add; the y and z
 * ghost zones hold the deposits that pm_fold_ghosts (or the slab exchange) adds to their owners. */
int pm_debug_buffer(pm_ctx *ctx, int channel, const double **dev_ptr, int64_t dims[3], int64_t *origin, int32_t *ghost);

/* Where pm_step_graph stands: 0 = the next call makes plain calls, 1 = the next call with the same arguments captures,
 * 2 = calls with the same arguments replay the graph.  HOST output. */
int pm_debug_graph_state(pm_ctx *ctx, int32_t *state);

/* Tiles of the buffer mesh (8^3 cells, ghost tiles included) and how many of them the last pm_deposit marked live per channel
 * group (K: accretion channel, N: supernova channels); stale tiles are neither reset nor read.  HOST outputs.  Synchronises. */
int pm_debug_tile_counts(pm_ctx *ctx, int64_t *n_tiles, int64_t *live_k, int64_t *live_n);

/* Return mesh: one record of 4 doubles per cell (eta of Eq. 4, pre-step velocity x, y, z), valid where buffer channel
 * 0 != 0.  *dev_ptr points at word `word` of cell 0; the same word of cell q is at dev_ptr[4 q]. */
int pm_debug_return_mesh(pm_ctx *ctx, int word, const double **dev_ptr);

/* PM_FLAG_REPRODUCIBLE only: apply the Appendix A rounding to the folded buffers in place (call after pm_fold_ghosts), so that
 * pm_debug_buffer shows the values the apply pass will use.  In the timed path the apply pass rounds the sums as it
 * reads them and the buffers keep the unrounded sums; the rounding is idempotent, so calling this first changes nothing. */
int pm_debug_round_buffers(pm_ctx *ctx);

/* lambda of Eq. 21 per cell (needs PM_FLAG_DEBUG_LAMBDA). */
int pm_debug_lambda(pm_ctx *ctx, const double **dev_ptr);

/* Per-particle scalars (need PM_FLAG_DEBUG_SCALARS), SoA with stride n:
 * sinks: 0 rho_inf, 1 v_inf, 2 c_inf, 3 r_BH, 4 mdot, 5 r_acc, 6 sum w, 7 member count
 * SNe:   0 M_snr, 1 V_snr, 2..4 v_COM, 5 n_H, 6 R_M, 7 |p_radial|, 8 regime (1 EJ, 2 ST, 3 MC) */
int pm_debug_sink_scalars(pm_ctx *ctx, const double **dev_ptr, int64_t *n);
int pm_debug_sn_scalars(pm_ctx *ctx, const double **dev_ptr, int64_t *n);

/* Stencil of ONE particle at (x,y,z), evaluated by the same device code the deposit uses.  kind 0 = sink: writes
 * 1 (member) / 0 for every cell of the (2g+1)^3 box; kind 1 = SN: writes the omega sub-sample count.  Box cells in
 * (k, j, i) order into dev_counts (DEVICE pointer, int32, >= (2g+1)^3 entries); host_ijk (HOST, 3 ints) receives
 * the host cell, *side (HOST) the box side.  Synchronises. */
int pm_debug_stencil(pm_ctx *ctx, int kind, double x, double y, double z, int32_t *dev_counts, int32_t *host_ijk,
                     int32_t *side);

#ifdef __cplusplus
}
#endif
#endif /* PM_B200_H */
