/*
 * sph.h -- C ABI of libsph.so: the data-parallel hot path of Gadget3's SPH modules on one B200.
 *
 * The paper states the problem, not an API: every module "compute[s] the force acting on a list of
 * active particles by performing a tree walk over groups of one or more active particles and find[s]
 * all neighbouring particles within a given distance" (§1); SPH is two such modules,
 * "the first one computes particle densities by multiple iterations and the second one computes
 * hydrodynamic forces" (§1).  The three calls below are that statement:
 * sph_build_index (the structure the neighbour search walks), sph_density (active list, neighbour
 * number target, tolerance) and sph_hydro_force (active list).  The SPH formulas themselves are the
 * readings R1..R16 of DESIGN.md (the paper prints none).
 *
 * Conventions
 *  - All array arguments are DEVICE pointers (caller-owned, e.g. torch tensors) unless the name ends
 *    in _host.  The library never frees or reallocates caller arrays; it writes only the entries of
 *    ACTIVE particles, indexed by the caller's particle id.  Sorted copies, the octree and scratch
 *    are private to the context.
 *  - Work is enqueued on the CUDA stream given to sph_create.  sph_build_index and sph_hydro_force are
 *    fully asynchronous; sph_density synchronises once (to return n_unconverged); sph_get_stats and the
 *    *_host entry points synchronise before returning.
 *  - Preconditions are checked on the device: 0 <= x < box for every coordinate (sph_build_index);
 *    active ids in [0, n) and listed once; 0 < H < box/2 and finite for the guesses of the active
 *    particles (sph_density) and for h of ALL particles (sph_hydro_force), whose rho must be > 0 and
 *    whose rho, omega, u, vel must be finite.  A call whose inputs violate one computes and writes
 *    NOTHING; the failure is sticky and is returned -- SPH_E_ARG, or SPH_E_HRANGE if the only
 *    violation is H >= box/2 -- by that call if it synchronises, else by the next synchronising call
 *    (sph_density, sph_get_stats, sph_step_host), which then computes nothing itself and clears it.
 *    Bad positions invalidate the index: every call reports them until sph_build_index is called again.
 *  - Geometry: periodic cube [0, box)^3, minimum-image distances, support radius H < box/2.
 *    H is the radius at which the kernel reaches zero (W = 0 for r >= H).
 *  - Errors are return codes (sph_status); no exceptions, no abort, no printing.  A sticky CUDA error
 *    is reported by every later call; sph_last_error describes the most recent failure.
 *  - There is no CPU fallback and no other backend: without a CUDA device every call that needs one
 *    returns SPH_E_CUDA.
 */
#ifndef SPH_H_
#define SPH_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sph_ctx sph_ctx; /* opaque; owns index + scratch only */

typedef enum {
    SPH_OK = 0,
    SPH_E_ARG = 1,      /* bad argument (NULL pointer, n < 0, unknown kernel, ...) */
    SPH_E_CUDA = 2,     /* CUDA runtime error (see sph_last_error) */
    SPH_E_NOINDEX = 3,  /* sph_density / sph_hydro_force before sph_build_index */
    SPH_E_OOM = 4,      /* device allocation failed */
    SPH_E_INTERNAL = 5, /* an internal capacity was exceeded (reported, never silent) */
    SPH_E_HRANGE = 6,   /* a support radius >= box / 2 (minimum image undefined) */
    SPH_W_NOCONV = 16   /* warning: some active particles stopped without |N - N_t| <= tol */
} sph_status;

enum { SPH_KERNEL_CUBIC = 0, SPH_KERNEL_WC6 = 1 };

/* per-particle status word written by sph_density: low 8 bits = evaluations used, then flags */
enum {
    SPH_ST_CONVERGED = 1 << 8, /* |N - N_t| <= tol at the returned H */
    SPH_ST_BRACKET = 1 << 9,   /* bracket [lo,hi] collapsed to 1e-6 relative (count jumps over the band) */
    SPH_ST_NOTCONV = 1 << 10,  /* max_iter evaluations used */
    SPH_ST_STALLED = 1 << 11   /* H pinned at the cap 0.49999 box */
};

typedef struct {
    int kernel;        /* SPH_KERNEL_CUBIC or SPH_KERNEL_WC6 (R1) */
    float box;         /* periodic cube edge L > 0 */
    float gamma;       /* adiabatic index (5/3) */
    float alpha_visc;  /* artificial viscosity alpha (1.0), R9 */
    int count_mode;    /* 0: kernel-weighted neighbour number drives the h iteration, 1: integer count (R2) */
    int max_iter;      /* cap on evaluations per particle (64); 1..255 */
    int group_cap;     /* max active particles per group (one warp per group); 0 = default; <= 32 */
    int group_node;    /* groups are cut from the highest octree nodes holding <= this many particles;
                          0 = default (2 * group_cap); raised to the leaf capacity (32) if smaller */
} sph_params;

typedef struct {
    int64_t n;                 /* particles in the index */
    int64_t n_nodes;           /* octree nodes */
    int64_t n_groups;          /* groups (leaf chunks) of the all-active case */
    int64_t launches;          /* kernels launched by this context so far (ours + CUB passes) */
    /* counters of the most recent sph_density call */
    int64_t dens_evals;        /* particle evaluations (sum over particles of iterations used) */
    int64_t dens_candidates;   /* distance tests */
    int64_t dens_pairs;        /* true pairs (r < H), self included */
    /* counters of the most recent sph_hydro_force call */
    int64_t force_candidates;
    int64_t force_pairs;       /* true pairs r < max(H_i,H_j), self excluded */
    /* device times (CUDA events on the context's stream) of the most recent calls, milliseconds */
    float t_index_ms;          /* sph_build_index: all kernels a1-a5 */
    float t_density_kernel_ms; /* the persistent gather + h-iteration kernel alone (a6-a9) */
    float t_force_prep_ms;     /* sorted force state + per-node max H (a9/a4 refresh) */
    float t_force_kernel_ms;   /* the hydro-force gather kernel alone (a10-a11) */
    int64_t node_pool_overflow; /* != 0: the octree node pool ran out during sph_build_index (extremely clumped input);
                                   some leaves then hold more than 32 particles -- results stay correct, the gather slows down */
} sph_stats;

/* Create a context. `cuda_stream` is a cudaStream_t (NULL = legacy default stream). */
int sph_create(sph_ctx **out, const sph_params *p, void *cuda_stream);
int sph_destroy(sph_ctx *ctx);

/*
 * Build the spatial index over n particles (steps a1-a5 of DESIGN.md): 48-bit Morton keys
 * (16 bits per axis), radix sort of (key, id), sorted float4 copy (x,y,z,m), inverse permutation,
 * an octree over the sorted order whose leaves hold <= 32 particles, and the group list: the highest
 * octree nodes holding <= group_node particles, each cut into balanced runs of <= group_cap consecutive
 * sorted particles (one warp per group).  Replaces the paper's Hilbert keys + domain decomposition +
 * tree build (PAPER.md:25, :41 §1, :194-196 §4).
 *   pos   [n*3] device, x,y,z per particle, 0 <= x < box (checked on the device, see Conventions);
 *   mass  [n] device or NULL; if NULL every particle has mass_scalar.
 * n = 0 is valid (later calls do nothing).  Asynchronous.  If the octree node pool runs out (more than
 * about two nodes per particle: extremely clumped input) the remaining cells stay oversize leaves: results
 * are unaffected, the gather slows down, and sph_stats.node_pool_overflow reports it.
 * Small sets are bound by the ~45 dependent kernel launches of the build: from the second call in a row with the same
 * (n, pos, mass, mass_scalar) on, the launch sequence is captured into a CUDA graph and replayed (same kernels, same
 * arguments, current contents of the arrays; not on the legacy default stream, which cannot be captured).
 */
int sph_build_index(sph_ctx *ctx, int64_t n, const float *pos, const float *mass, float mass_scalar);

/*
 * Refresh the index after the particles have MOVED A LITTLE (same n, same ids): the sorted order, the octree and the
 * groups of the last sph_build_index are kept, the sorted positions are replaced by the new ones and every octree cell
 * is enlarged by the distance its farthest particle now lies outside it.  Results of the later calls are exactly those
 * of a fresh build (the neighbour search only prunes more conservatively), at about a fifth of its cost; the pruning
 * degrades as particles stray from their cells, so rebuild once displacements become comparable to the support radii.
 * This is what keeps time-steps with few active particles cheap (PAPER.md:57 §2, :86 §2.2, :160 §3.3: the paper's weak
 * point; SURVEY.md §8(f)-3 "incremental index refresh instead of full rebuild").  pos [n*3] device, 0 <= x < box
 * (checked on the device).  Asynchronous.
 */
int sph_refresh_index(sph_ctx *ctx, int64_t n, const float *pos);

/*
 * SPH density with the smoothing-length iteration (steps a5-a9; R1-R7):
 * for every active particle, starting from h[id], iterate the safeguarded Newton rule of R7 on the
 * support radius until the neighbour number N (kernel-weighted, or integer with count_mode 1)
 * satisfies |N - n_ngb_target| <= n_ngb_tol, then write
 *   h[id]         converged support radius,
 *   rho[id]       sum_j m_j W(r_ij, H_i)  (self term included),
 *   omega[id]     1 + (H_i / 3 rho_i) d rho_i / d H_i,
 *   ngb_count[id] integer count #{j : r_ij < H_i} at the returned H (self included),
 *   status[id]    evaluations used | SPH_ST_* flags (status may be NULL).
 *   active        [n_active] device int32 particle ids (in range, each listed once); NULL with n_active != 0
 *                 (conventionally -1) means all particles; n_active == 0 is the empty list (nothing
 *                 is computed or written, whatever the pointer);
 *   n_ngb_tol     +inf means "evaluate once at the given h";
 *   n_unconverged_host  HOST pointer (may be NULL): number of active particles that stopped
 *                 without SPH_ST_CONVERGED.
 * Returns SPH_OK, or SPH_W_NOCONV if *n_unconverged_host would be > 0.  Synchronises once.
 * A failed precondition (ids, guesses; see Conventions) makes the call compute and write nothing and
 * return SPH_E_ARG / SPH_E_HRANGE.
 */
int sph_density(sph_ctx *ctx, const int32_t *active, int64_t n_active, float n_ngb_target, float n_ngb_tol,
                float *h, float *rho, float *omega, int32_t *ngb_count, int32_t *status,
                int64_t *n_unconverged_host);

/*
 * Symmetric SPH hydro-force pair sum (steps a5, a6, a10, a11; R8-R12): for every active
 * particle i, over all j != i with r_ij < max(H_i, H_j),
 *   acc[id*3..]  = - sum_j m_j [A_i F_ij(H_i) + A_j F_ij(H_j) + Pi_ij Fbar_ij] rhat_ij
 *   dudt[id]     =   sum_j m_j [A_i F_ij(H_i) + Pi_ij Fbar_ij / 2] (v_ij . rhat_ij)
 *   vsig_max[id] =   max_j (c_i + c_j - 3 min(0, v_ij . rhat_ij))     (0 if no neighbour)
 * with A = (gamma-1) u / (omega rho), F_ij(H) = dW/dr(r_ij, H), Pi_ij the signal-velocity viscosity.
 *   vel [n*3], u [n], h [n], rho [n], omega [n]: device, valid for ALL n particles (inactive
 *   neighbours contribute with their current values, R12); acc [n*3], dudt [n], vsig_max [n]: device,
 *   written for active particles only.  Asynchronous: a failed precondition (ids, h, rho, ...; see
 *   Conventions) makes the call compute and write nothing, and the next synchronising call
 *   (sph_density, sph_get_stats) returns SPH_E_ARG / SPH_E_HRANGE instead of doing its own work.
 */
int sph_hydro_force(sph_ctx *ctx, const int32_t *active, int64_t n_active, const float *vel, const float *u,
                    const float *h, const float *rho, const float *omega, float *acc, float *dudt,
                    float *vsig_max);

/*
 * Improved-SPH extension: the SPH flavour the paper's runs use is "the improved SPH
 * of ref [6]" (PAPER.md:25 §1, :209), which the paper only cites; readings R17-R20.
 *
 * sph_velocity_gradients -- R17, a third gather over the same index: for every active particle i, over
 * j != i with r_ij < H_i (its own support),
 *   divv[id]       = (1/rho_i) sum_j m_j (v_j - v_i) . grad_i W_ij(H_i)
 *   curlv[id*3..]  = (1/rho_i) sum_j m_j (v_i - v_j) x grad_i W_ij(H_i),  grad_i W_ij = dW/dr(r_ij, H_i) rhat_ij.
 * vel [n*3], h [n], rho [n] device, valid for all particles; divv [n], curlv [n*3] written for active
 * particles only.  Asynchronous; preconditions and error reporting as sph_hydro_force.
 *
 * sph_hydro_force_improved -- sph_hydro_force with
 *   R19 a per-particle viscosity coefficient: Pi_ij uses (alpha_i + alpha_j)/2 in place of alpha_visc, and
 *       dalpha_dt[id] = -(alpha_i - alpha_min) 2 l c_i / H_i + max(0, -div v_i)(alpha_max - alpha_i);
 *   R18 the shear limiter f_i = |div v_i| / (|div v_i| + |curl v_i| + 1e-4 c_i / H_i) (if balsara != 0):
 *       Pi_ij is multiplied by (f_i + f_j)/2;
 *   R20 artificial conduction: dudt += sum_j m_j alpha_cond sqrt(|P_i - P_j| / rho_ij) (u_i - u_j) Fbar_ij / rho_ij.
 * alpha [n], divv [n], curlv [n*3]: device, valid for ALL particles (neighbours contribute with theirs).
 */
typedef struct {
    float alpha_min;   /* floor of the viscosity coefficient (0.02) */
    float alpha_max;   /* its ceiling (3.0) */
    float decay_l;     /* decay length l of R19 (4.0) */
    float alpha_cond;  /* artificial conduction coefficient (0.25); 0 switches conduction off */
    int balsara;       /* shear limiter on / off */
} sph_improved_params;

int sph_velocity_gradients(sph_ctx *ctx, const int32_t *active, int64_t n_active, const float *vel, const float *h,
                           const float *rho, float *divv, float *curlv);
int sph_hydro_force_improved(sph_ctx *ctx, const int32_t *active, int64_t n_active, const float *vel, const float *u,
                             const float *h, const float *rho, const float *omega, const float *alpha, const float *divv,
                             const float *curlv, const sph_improved_params *ip, float *acc, float *dudt, float *vsig_max,
                             float *dalpha_dt);

/*
 * Thermal conduction: the paper's third module of the same pattern (PAPER.md:27 §1, :41, :102
 * §2.4, :156 §3.3; no equations given) as a further pair pass over the same index; reading R21.  For every
 * active particle i, over j != i with r_ij < max(H_i, H_j),
 *   dudt_cond[id] = sum_j m_j / (rho_i rho_j) * [4 k_i k_j / (k_i + k_j)] * (u_i - u_j) * Fbar_ij / r_ij,
 *   k = kappa0 * u^kappa_exp   (kappa_exp = 2.5: Spitzer; 0: constant conductivity; T = u up to constants in kappa0).
 * u [n], h [n], rho [n]: device, valid for all particles; dudt_cond [n] written for active particles only.
 * Asynchronous; preconditions and error reporting as sph_hydro_force.
 */
int sph_thermal_conduction(sph_ctx *ctx, const int32_t *active, int64_t n_active, const float *u, const float *h,
                           const float *rho, float kappa0, float kappa_exp, float *dudt_cond);

/*
 * Short-range Barnes-Hut gravity on the octree of the index (SURVEY.md §8(f)-4; PAPER.md:25 §1, :41, :102-104 §2.4;
 * DESIGN.md reading R23): for every active particle i
 *   acc_grav[id*3..] = - G sum_{j != i, r < r_cut} m_j d_ij / (r^2 + eps^2)^(3/2) [erfc(r / 2 r_s) + r / (r_s sqrt(pi)) exp(-r^2 / 4 r_s^2)],
 * the short-range force of a TreePM split, evaluated with a grouped tree walk: a cell whose edge is smaller than theta
 * times the distance from the group's bounding box to the cell's centre of mass enters as ONE pseudo-particle
 * (monopole), closer cells are opened down to their particles.  theta = 0 opens everything: the exact direct sum.
 * Uses the positions and masses of the index only.  r_cut < box/2.  acc_grav [n*3] device, written for active particles.
 * Asynchronous.
 */
int sph_gravity_short(sph_ctx *ctx, const int32_t *active, int64_t n_active, float G, float r_s, float r_cut, float eps,
                      float theta, float *acc_grav);

/*
 * Kick-drift-kick time integration with power-of-two time bins (SURVEY.md §8(f)-3; PAPER.md:37 §1, :84-86 §2.2, :114
 * §3: the scheme that produces the paper's active lists, down to "one or very few" particles per step; no formulas in
 * the paper: DESIGN.md reading R22).  Timeline of T = 2^(n_bins-1) ticks per dt_max; a particle of bin b steps
 * dt_max / 2^b.  Time-step criterion dt_i = min(courant * H_i / vsig_i, sqrt(2 eta H_i / |a_i|)), bin = smallest b with
 * dt_max / 2^b <= dt_i; a particle may move to a longer step one bin at a time and only where the timeline is aligned.
 *   sph_kdk_init: tick 0 -- index, density and force for all particles, bins, first half kick (vel, u become
 *                 kick-centred).  h is the guess on entry.
 *   sph_kdk_step: advance to the next tick at which a step ends; drift ALL particles there (pos, periodic wrap;
 *                 vpred, upred = velocity and energy extrapolated to that time with the stored acc, dudt); the
 *                 particles whose step ends are active: sph_build_index -- or, for a step with fewer than
 *                 rebuild_fraction * n active particles and at most refresh_max times in a row, sph_refresh_index (the
 *                 same results, see there) --, sph_density (last h as the guess), sph_hydro_force (with vpred, upred)
 *                 on them; second half kick, new bin, first half kick.
 *                 *tick_host = the new tick, *n_active_host = number of active particles (their ids, ascending,
 *                 are left in state->active).  Synchronises.
 * All arrays of sph_kdk_state are DEVICE arrays owned by the caller.
 */
typedef struct {
    float dt_max;       /* length of the longest step (bin 0) */
    int n_bins;         /* 1..24 */
    float courant;      /* 0.3 */
    float eta;          /* 0.025 */
    float n_ngb_target, n_ngb_tol;
    int refresh_max;    /* steps in a row that may refresh the index instead of rebuilding it; 0 = always rebuild */
    float rebuild_fraction; /* rebuild whenever n_active >= rebuild_fraction * n (1/16) */
    /* grav_G > 0: the short-range gravity of sph_gravity_short (same parameters) is added to the hydro acceleration of
     * the active particles; the time-step criterion sees the sum.  grav_G = 0: hydrodynamics only. */
    float grav_G, grav_rs, grav_rcut, grav_eps, grav_theta;
} sph_kdk_params;

typedef struct {
    float *pos;         /* n*3 */
    float *vel;         /* n*3, kick-centred after sph_kdk_init */
    float *u, *h, *rho, *omega; /* n each */
    int32_t *ngb;       /* n */
    float *acc;         /* n*3 */
    float *dudt, *vsig; /* n each */
    float *vpred;       /* n*3 */
    float *upred;       /* n */
    int32_t *bin, *tbegin, *active; /* n each: time bin, tick at which the current step began, active list */
} sph_kdk_state;

int sph_kdk_init(sph_ctx *ctx, int64_t n, float mass_scalar, const sph_kdk_params *p, const sph_kdk_state *state);
int sph_kdk_step(sph_ctx *ctx, int64_t n, float mass_scalar, const sph_kdk_params *p, const sph_kdk_state *state,
                 int64_t *tick_host, int64_t *n_active_host);

/*
 * One whole pass of the hot path with HOST buffers (used for the end-to-end measurement): copies
 * pos, vel, u, h (guess) [and active ids] to the device, runs sph_build_index, sph_density and
 * sph_hydro_force, copies h, rho, omega, ngb_count, acc, dudt, vsig_max back -- the whole arrays when all
 * particles are active; with an active list only the active particles' entries travel (packed on the device,
 * 36 bytes each) and the other entries of the caller's arrays are left as they are --, and synchronises.  All pointers are HOST pointers;
 * `active_host` may be NULL (all active).  With PINNED host memory the copies overlap the kernels on a
 * second stream of the context: h, vel and u go up while the index is built and the density runs, h, rho,
 * omega and ngb_count come down while the force pass runs; only pos (up) and acc, dudt, vsig_max (down)
 * are exposed.  With pageable memory the copies are staged by the driver and the call is merely slower.
 */
int sph_step_host(sph_ctx *ctx, int64_t n, const float *pos_host, const float *vel_host, const float *u_host,
                  float mass_scalar, const int32_t *active_host, int64_t n_active, float n_ngb_target,
                  float n_ngb_tol, float *h_host /* in: guess, out */, float *rho_host, float *omega_host,
                  int32_t *ngb_count_host, float *acc_host, float *dudt_host, float *vsig_host,
                  int64_t *n_unconverged_host);

/*
 * Stream compaction of 0/1 flags: ids_out[k] = index of the k-th non-zero flag, ascending (k < count), *count_dev =
 * their number -- the step that turns per-particle "my time-step ends now" flags into the active list of the next
 * call (§2.2: the active particles of a time bin; it is what sph_kdk_step does inside).  flags [n] u32
 * (0 or 1), ids_out [n] i32 (entries from count on are left as they were), count_dev [1] u32: DEVICE arrays owned by
 * the caller.  Asynchronous on the context's stream; n < 2^31.
 *   sph_compact_flags          block sums in the context's scratch buffer, which grows by cudaFree + cudaMalloc when n
 *                              exceeds every earlier call's.
 *   sph_compact_flags_noalloc  the same kernels, same results, for callers that must not allocate (code under CUDA graph
 *                              capture, serving loops, harnesses that forbid it): the block sums live in a fixed array
 *                              of 64 KB of device memory that every GPU loading the library holds until exit.  The call
 *                              launches kernels and nothing else: no cudaMalloc, cudaFree or allocating library routine
 *                              (the very first call on a device also asks the runtime for the array's address).
 *                              n > SPH_COMPACT_NOALLOC_MAX is rejected with SPH_E_ARG and a message.  All calls on a
 *                              device share the array, whichever context or stream they use: calls that may overlap on
 *                              the GPU (different streams, no ordering between them) race and give wrong results;
 *                              calls ordered on one stream are safe, and nothing of an earlier call is read by a later one.
 */
#define SPH_COMPACT_NOALLOC_MAX 67108864 /* 2^26 flags */
int sph_compact_flags(sph_ctx *ctx, int64_t n, const uint32_t *flags, int32_t *ids_out, uint32_t *count_dev);
int sph_compact_flags_noalloc(sph_ctx *ctx, int64_t n, const uint32_t *flags, int32_t *ids_out, uint32_t *count_dev);

/* Counters of the last calls (host struct filled; synchronises the stream).  Reports a pending
 * precondition failure of an earlier asynchronous call (see Conventions). */
int sph_get_stats(sph_ctx *ctx, sph_stats *out_host);

/* Text of the most recent error of this context ("" if none). Never NULL; valid until the next call. */
const char *sph_last_error(const sph_ctx *ctx);

/* Library version string and the compute capability it was built for ("sm_100a"). */
const char *sph_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SPH_H_ */
