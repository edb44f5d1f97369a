// sph_internal.cuh -- private declarations of libsph.so (CUDA path; shares nothing with oracle/).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "sph.h"

#ifdef SPH_DEBUG
#include <assert.h>
#define SPH_ASSERT(c) assert(c)
#else
#define SPH_ASSERT(c) ((void)0)
#endif

#define SPH_LMAX 16         // octree depth: 16 bits per axis -> 48-bit Morton keys
#define SPH_KEY_BITS (3 * SPH_LMAX)
#ifndef SPH_LEAF
#define SPH_LEAF 32         // octree leaf capacity (a candidate segment is a run of sibling leaves)
#endif
#define SPH_MAXB 32         // max actives per group (a warp: one lane per active and stream)
#define SPH_GCAP_DEFAULT 8  // default actives per group (leaves are cut into balanced runs)
#ifndef SPH_WARPS
#define SPH_WARPS 4         // warps per CTA of the gather kernels (warps are independent)
#endif
#define SPH_THREADS (32 * SPH_WARPS)
#ifndef SPH_CTAS
#define SPH_CTAS 5          // resident CTAs per SM the gather kernels are compiled for (register budget)
#endif
#define SPH_SMAX 128        // candidate segments per walk batch (per warp)
#define SPH_STK 192         // walk stack entries (blocks of 8 sibling nodes, per warp)
#define SPH_STK4 48         // 4-block pops only while the stack is at most this deep
#define SPH_CH 120          // candidates per chunk (60 pairs: divisible by 1..6, 10, 12, 15, 20, 30)
#ifndef SPH_CTAS_FORCE
#define SPH_CTAS_FORCE SPH_CTAS
#endif
#ifndef SPH_QCAP
#define SPH_QCAP 32         // per-lane hit-queue entries (>= 2 * SPH_QSTEP)
#endif
#ifndef SPH_QCAP_FORCE
#define SPH_QCAP_FORCE 48   // the same for the force kernel (a hit costs ~95 instructions there: fuller drains pay;
                            // measured at C4: 32 -> 75.1 ms, 44 -> 73.0, 48 -> 72.8, 52 -> 72.7, 64 (4 CTAs per SM) -> 83.0)
#endif
#ifndef SPH_QSTEP_FORCE
#define SPH_QSTEP_FORCE 15  // the same for the force kernel (12 and 20 measured equal or slower)
#endif
#ifndef SPH_QSTEP
#define SPH_QSTEP 15        // candidate-pair steps (2 tests each) between queue-capacity checks
#endif
#define SPH_NA 1            // actives per lane of the density gather (2 measured slower: profiles/r1j_gather.md)
#define SPH_GBLOCK 1        // consecutive groups a warp takes per work-counter increment (1: shortest tail, measured)

// device-side precondition failures (SphCounters::err / idx_err)
#define SPH_ERR_IDS 1u      // an active id outside [0, n)
#define SPH_ERR_DUP 2u      // an active id listed twice
#define SPH_ERR_H 4u        // a support radius <= 0 or not finite (guess of sph_density, h of sph_hydro_force)
#define SPH_ERR_HRANGE 8u   // a support radius >= box / 2
#define SPH_ERR_STATE 16u   // rho <= 0 or rho / omega / u / vel not finite in sph_hydro_force
#define SPH_ERR_POS 32u     // a coordinate outside [0, box) or not finite in sph_build_index

// octree node, 32 bytes, read as two 16-byte loads
struct __align__(16) SphNode {
    uint32_t start;   // first sorted slot
    uint32_t count;   // particles in the cell
    uint32_t child;   // index of the first of 8 consecutive children, 0 = leaf
    uint32_t parent;  // parent node index (root: 0)
    float cx, cy, cz; // cell centre
    float half;       // half edge
};

// device-side counters, one block of unsigned ints / 64-bit
struct SphCounters {
    unsigned int n_nodes;
    unsigned int n_groups;     // all-active groups
    unsigned int n_agroups;    // groups of the current active subset
    unsigned int overflow;     // node pool exhausted (graceful: oversize leaves)
    unsigned int work;         // persistent-kernel group counter
    unsigned int n_unconv;     // density: particles stopped without convergence
    unsigned int err;          // SPH_ERR_* bits of the calls since the last report: sticky, the gather kernels compute
                               // nothing while it is set; the next synchronising call reports and clears it
    unsigned int idx_err;      // SPH_ERR_POS: state of the current index (cleared by the next sph_build_index)
    unsigned int lvl_begin[SPH_LMAX + 3];
    unsigned int lvl_done[SPH_LMAX + 3];
    unsigned long long dens_evals, dens_cands, dens_pairs, force_cands, force_pairs;
};

struct sph_ctx {
    sph_params prm;
    cudaStream_t stream;
    char err[320];
    int device_sms;
    int64_t n;        // particles in the index
    int64_t cap_n;    // allocated capacity (particles)
    bool have_index;
    bool has_mass;
    float mass_scalar;
    int grp_cap;      // max actives per group
    int grp_node;     // groups are cut from the highest octree nodes holding <= this many particles

    // index (device)
    uint64_t *keys, *keys_alt;
    uint32_t *perm, *perm_alt, *inv;
    float4 *xyzm;
    SphNode *nodes;
    int64_t node_cap;
    uint32_t *grp_mark, *gid_of_slot, *grp_start;
    uint32_t *slot_leaf;  // octree leaf of every sorted slot
    SphCounters *cnt;
    uint32_t *sort_hist;   // radix sort: per-tile digit histograms + digit bases
    size_t sort_cap;
    uint32_t *scan_bsum;   // scan: block sums
    size_t scan_cap;

    // force pass (device)
    float4 *f_xyzh, *f_vc, *f_ext; // f_ext: improved-SPH record (alpha, f, u), allocated on first use
    float *node_hmax;
    bool act_keep;        // sph_active_groups: keep the groups of the last call (set by sph_kdk_step / sph_step_* between density and force)
    float *kdk_grav;      // sph_kdk_*: gravity of the active particles before it is added to acc
    int64_t kdk_grav_cap;
    int kdk_refreshed;    // steps of sph_kdk_step since the last full build
    float *node_slack;    // sph_refresh_index: how far particles have left their cells (per node)
    float4 *node_mom;     // short-range gravity: centre of mass and mass of every node (allocated on first use)
    int64_t node_mom_cap;

    // active subset scratch (device)
    int64_t cap_act;
    uint32_t *act_slot, *act_slot_alt, *act_flag, *agrp_start;

    // host-step device state
    int64_t cap_host;
    float *d_pos, *d_vel, *d_u, *d_h, *d_rho, *d_omega, *d_acc, *d_dudt, *d_vsig;
    int32_t *d_ngb, *d_active;
    uint32_t *d_pack, *h_pack;   // sph_step_host with an active list: the actives' results packed (device / pinned host), 9 words each
    int64_t cap_pack;

    int64_t launches;
    int64_t kdk_tick;  // sph_kdk_*: current tick of the integer timeline

    // phase timing: events recorded on the stream around the phases named in sph_stats
    cudaEvent_t ev[8]; // 0,1 index  2,3 density kernel  4,5 force prep  6,7 force kernel
    // sph_build_index, launch-bound for small sets (~45 dependent launches): the second call in a row with the same
    // (n, pos, mass, mass_scalar) captures the launch sequence into a CUDA graph, later ones replay it (not on the legacy
    // default stream, which cannot be captured)
    cudaGraphExec_t idx_graph;
    const float *gk_pos, *gk_mass; // key of the graph (idx_graph != NULL) ...
    const float *lk_pos, *lk_mass; // ... and of the last direct build
    int64_t gk_n, lk_n;
    float gk_ms, lk_ms;
    int64_t idx_graph_launches;
    bool idx_graph_off;            // capture failed once: stay with direct launches
    cudaStream_t copy_stream; // sph_step_host: host copies that overlap the kernels (created at first use)
    cudaEvent_t cev[4];       // sph_step_host: positions up / velocities, energies up / density results final / h up
    bool ev_set[4];
};

// error helpers -------------------------------------------------------------------------------
int sph_fail(sph_ctx *ctx, int code, const char *fmt, ...);
#define SPH_CUDA(ctx, call)                                                                          \
    do {                                                                                             \
        cudaError_t e_ = (call);                                                                     \
        if (e_ != cudaSuccess)                                                                       \
            return sph_fail(ctx, e_ == cudaErrorMemoryAllocation ? SPH_E_OOM : SPH_E_CUDA,           \
                            "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__);    \
    } while (0)

// pair physics of the force gather kernel (sph_force_launch)
enum { SPH_MODE_BASE = 0, SPH_MODE_IMPROVED = 1, SPH_MODE_GRADV = 2, SPH_MODE_CONDUCT = 3 };

// stages (each returns sph_status) --------------------------------------------------------------
int sph_index_build(sph_ctx *ctx, const float *pos, const float *mass);
int sph_index_refresh(sph_ctx *ctx, const float *pos);
int sph_active_reserve(sph_ctx *ctx, int64_t cap);
int sph_gravity_launch(sph_ctx *ctx, bool subset, int64_t n_items, float G, float r_s, float r_cut, float eps, float theta, float *acc);
// stable LSD radix sort on the low `bits` key bits; *in_alt = 1 if the result ended up in the *_alt buffers
int sph_sort_pairs_u64(sph_ctx *ctx, uint64_t *keys, uint64_t *keys_alt, uint32_t *vals, uint32_t *vals_alt, int64_t n, int bits,
                       int *in_alt);
int sph_sort_keys_u32(sph_ctx *ctx, uint32_t *keys, uint32_t *keys_alt, int64_t n, int bits, int *in_alt);
// inclusive scan of 0/1 marks (incl may be NULL) + positions of the marks (start) + their number (*count_dev, device)
int sph_scan_marks(sph_ctx *ctx, const uint32_t *mark, int64_t n, uint32_t *incl, uint32_t *start, unsigned int *count_dev);
void sph_reset_counters(sph_ctx *ctx, int which, bool subset); // 0: density, 1: force
int sph_active_groups(sph_ctx *ctx, const int32_t *active, int64_t n_active);
int sph_density_launch(sph_ctx *ctx, const int32_t *active, int64_t n_items, float n_target, float n_tol, float *h,
                       float *rho, float *omega, int32_t *ngb, int32_t *status);
int sph_force_launch(sph_ctx *ctx, int mode, bool subset, int64_t n_items, const float *vel, const float *u, const float *h,
                     const float *rho, const float *omega, float *acc, float *dudt, float *vsig, const float *alpha,
                     const float *divv, const float *curlv, const sph_improved_params *ip, float *dalpha, float *divv_out,
                     float *curlv_out, float kappa0 = 0.f, float kappa_exp = 0.f);
