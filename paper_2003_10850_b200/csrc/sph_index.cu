// sph_index.cu -- steps a1-a5: Morton keys, radix sort, permute to sorted float4, octree over the
// sorted order, group (leaf-chunk) lists for the all-active and the active-subset case.
//
// Replaces the paper's Hilbert keys + domain decomposition + serial tree build (§1,
// :72 §2.1, :194-196 §4) and its N_min CPU fallback for small active sets (§2.2).
#include <stddef.h>

#include <algorithm>

#include "sph_internal.cuh"

namespace {

// interleave 16 bits with two zero bits between consecutive bits
__device__ __forceinline__ uint64_t part1by2_16(uint32_t v)
{
    uint64_t x = v & 0xffffu;
    x = (x | (x << 16)) & 0x00000000ff0000ffull;
    x = (x | (x << 8)) & 0x000000f00f00f00full;
    x = (x | (x << 4)) & 0x00000c30c30c30c3ull;
    x = (x | (x << 2)) & 0x0000249249249249ull;
    return x;
}

__device__ __forceinline__ uint32_t cell16(float x, float scale)
{
    int c = __float2int_rd(x * scale);
    c = max(0, min(c, (1 << SPH_LMAX) - 1));
    return (uint32_t)c;
}

// a1: key generation
__global__ void k_keys(int64_t n, const float *__restrict__ pos, float scale, float box, uint64_t *__restrict__ keys,
                       uint32_t *__restrict__ perm, SphCounters *cnt)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
    // precondition 0 <= x < box (also catches NaN): the index is marked unusable, every later call reports it
    if (!(x >= 0.f && x < box && y >= 0.f && y < box && z >= 0.f && z < box)) atomicOr(&cnt->idx_err, SPH_ERR_POS);
    uint64_t k = part1by2_16(cell16(x, scale)) | (part1by2_16(cell16(y, scale)) << 1) |
                 (part1by2_16(cell16(z, scale)) << 2);
    keys[i] = k;
    perm[i] = (uint32_t)i;
}

// a3: gather into the sorted float4 copy, inverse permutation
__global__ void k_permute(int64_t n, const float *__restrict__ pos, const float *__restrict__ mass, float mass_scalar,
                          const uint32_t *__restrict__ perm, float4 *__restrict__ xyzm, uint32_t *__restrict__ inv)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t id = perm[i];
    float4 p;
    p.x = pos[3 * (int64_t)id];
    p.y = pos[3 * (int64_t)id + 1];
    p.z = pos[3 * (int64_t)id + 2];
    p.w = mass ? mass[id] : mass_scalar;
    xyzm[i] = p;
    inv[id] = (uint32_t)i;
}

__global__ void k_tree_init(SphCounters *cnt, SphNode *nodes, uint32_t n, float box)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        SphNode r;
        r.start = 0; r.count = n; r.child = 0; r.parent = 0;
        r.cx = r.cy = r.cz = 0.5f * box; r.half = 0.5f * box;
        nodes[0] = r;
        cnt->n_nodes = 1;
        cnt->overflow = 0;
        cnt->n_groups = 0;
        for (int l = 0; l < SPH_LMAX + 3; l++) { cnt->lvl_begin[l] = 1; cnt->lvl_done[l] = 0; }
        cnt->lvl_begin[0] = 0;
        cnt->lvl_begin[1] = 1;
    }
}

// a4: split every node of `level` that holds more than leaf_cap particles into its 8 octants.
// The octant of a particle at this level is a 3-bit digit of its key; the sorted order makes each
// child a contiguous run found by binary search.  Eight lanes share a node: lane k finds the start of
// octant k, so the seven dependent-load chains of a node run side by side (the kernel is bound by
// that latency at the top levels, where a run holds millions of keys).
__global__ void k_tree_split(SphCounters *cnt, SphNode *nodes, const uint64_t *__restrict__ keys, int level,
                             uint32_t leaf_cap, uint32_t node_cap)
{
    const uint32_t beg = cnt->lvl_begin[level], end = cnt->lvl_begin[level + 1];
    const int shift = 3 * (SPH_LMAX - 1 - level);
    const uint32_t k = threadIdx.x & 7u;
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, nthr = gridDim.x * blockDim.x;
    // warp-uniform trip count: a warp covers 4 consecutive nodes per step
    for (uint32_t base = beg + ((tid & ~31u) >> 3); base < end; base += nthr >> 3) {
        const uint32_t nd = base + ((threadIdx.x & 31u) >> 3);
        const bool valid = nd < end;
        SphNode p = nodes[valid ? nd : beg];
        const bool split = valid && p.count > leaf_cap;
        uint32_t c0 = 0;
        if (split && k == 0) c0 = atomicAdd(&cnt->n_nodes, 8u);
        c0 = __shfl_sync(0xffffffffu, c0, threadIdx.x & 24u);
        const bool ok = split && c0 + 8u <= node_cap;
        if (split && !ok && k == 0) atomicExch(&cnt->overflow, 1u); // stays an oversize leaf
        // first slot in [start, start + count) whose digit >= k
        uint32_t lo = p.start, hi = p.start + p.count;
        if (!ok || k == 0) hi = lo;
        while (lo < hi) {
            const uint32_t mid = lo + ((hi - lo) >> 1);
            const uint32_t dig = (uint32_t)(keys[mid] >> shift) & 7u;
            if (dig < k) lo = mid + 1; else hi = mid;
        }
        uint32_t nxt = __shfl_down_sync(0xffffffffu, lo, 1);
        if (k == 7u) nxt = p.start + p.count;
        if (ok) {
            const float q = 0.5f * p.half;
            SphNode c;
            c.start = lo; c.count = nxt - lo; c.child = 0; c.parent = nd;
            c.cx = p.cx + ((k & 1) ? q : -q);
            c.cy = p.cy + ((k & 2) ? q : -q);
            c.cz = p.cz + ((k & 4) ? q : -q);
            c.half = q;
            nodes[c0 + k] = c;
            if (k == 0) nodes[nd].child = c0;
        }
    }
    // last block to finish publishes the end of the next level
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        unsigned int t = atomicAdd(&cnt->lvl_done[level], 1u);
        if (t == gridDim.x - 1) {
            __threadfence();
            unsigned int nn = atomicAdd(&cnt->n_nodes, 0u);
            if (nn > node_cap) { nn = node_cap - ((node_cap - 1) & 7u); cnt->n_nodes = nn; }
            cnt->lvl_begin[level + 2] = nn;
        }
    }
}

// a5 (all-active case): the group nodes are the highest octree nodes that hold <= node_cap particles
// (a leaf that holds more, e.g. coincident particles, is its own group node); every group node is cut
// into ceil(count / grp_cap) balanced runs of consecutive sorted slots; a run is a group (consecutive
// Morton order inside a small cell keeps a run spatially compact)
// (+ the leaf of every sorted slot, for the per-particle passes that feed per-node maxima: k_force_prep, k_refresh_slots)
__global__ void k_mark_groups(const SphCounters *cnt, const SphNode *__restrict__ nodes, uint32_t grp_cap,
                              uint32_t node_cap, uint32_t *__restrict__ mark, uint32_t *__restrict__ slot_leaf)
{
    uint32_t nn = cnt->n_nodes;
    for (uint32_t nd = blockIdx.x * blockDim.x + threadIdx.x; nd < nn; nd += gridDim.x * blockDim.x) {
        SphNode p = nodes[nd];
        if (p.child == 0)
            for (uint32_t s = 0; s < p.count; s++) slot_leaf[p.start + s] = nd;
        if (p.count == 0 || (p.count > node_cap && p.child != 0)) continue;
        if (nd != 0 && nodes[p.parent].count <= node_cap) continue; // an ancestor is the group node
        const uint32_t ns = (p.count + grp_cap - 1) / grp_cap;
        for (uint32_t s = 0; s < ns; s++) mark[p.start + (uint32_t)(((uint64_t)s * p.count) / ns)] = 1u;
    }
}

__global__ void k_act_slots(int64_t na, int64_t n, const int32_t *__restrict__ active, const uint32_t *__restrict__ inv,
                            uint32_t *__restrict__ slot, SphCounters *cnt)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= na) return;
    const int32_t id = active[k];
    const bool ok = id >= 0 && (int64_t)id < n;
    if (!ok) atomicOr(&cnt->err, SPH_ERR_IDS); // the gather kernels then return at once; reported as SPH_E_ARG
    slot[k] = ok ? inv[id] : 0u;
}

__global__ void k_act_flags(int64_t na, const uint32_t *__restrict__ slot, const uint32_t *__restrict__ gid,
                            uint32_t *__restrict__ flag, SphCounters *cnt)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= na) return;
    flag[k] = (k == 0 || gid[slot[k]] != gid[slot[k - 1]]) ? 1u : 0u;
    // an id listed twice sits next to itself in the sorted slots (and would make a group larger than a warp)
    if (k > 0 && slot[k] == slot[k - 1] && !(cnt->err & SPH_ERR_IDS)) atomicOr(&cnt->err, SPH_ERR_DUP);
}

// ---- sph_refresh_index: the particles moved a little since the build; keep the tree, make every cell large enough ----
__device__ __forceinline__ int level_of(const SphCounters *cnt, uint32_t nd)
{
    int l = 0;
    while (l < SPH_LMAX && nd >= cnt->lvl_begin[l + 1]) l++;
    return l;
}

// every sorted slot: fetch the particle's new position into the sorted copy; slack of its leaf = how far the farthest of
// the leaf's particles now lies outside the leaf's cell (periodic), handed up the parent chain (a particle outside a
// cell by s is outside each ancestor's cell by at most s).  The lanes of a warp that share a leaf send one value.
__global__ void k_refresh_slots(int64_t n, SphCounters *cnt, const SphNode *__restrict__ nodes, const uint32_t *__restrict__ perm,
                                const uint32_t *__restrict__ slot_leaf, const float *__restrict__ pos, float box,
                                float4 *__restrict__ xyzm, float *__restrict__ slack)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool in = i < n;
    uint32_t leaf = 0xffffffffu;
    float d = 0.f;
    if (in) {
        const uint32_t id = perm[i];
        const float x = pos[3 * (size_t)id], y = pos[3 * (size_t)id + 1], z = pos[3 * (size_t)id + 2];
        if (!(x >= 0.f && x < box && y >= 0.f && y < box && z >= 0.f && z < box)) atomicOr(&cnt->idx_err, SPH_ERR_POS);
        float4 q = xyzm[i];
        q.x = x; q.y = y; q.z = z;
        xyzm[i] = q;
        leaf = slot_leaf[i];
        const SphNode p = nodes[leaf];
        float dx = fabsf(x - p.cx), dy = fabsf(y - p.cy), dz = fabsf(z - p.cz);
        dx = fminf(dx, box - dx); dy = fminf(dy, box - dy); dz = fminf(dz, box - dz);
        d = fmaxf(fmaxf(dx, dy), dz); // >= 0 (NaN -> 0: the position error is already recorded)
    }
    const unsigned grp = __match_any_sync(0xffffffffu, leaf);
    const int db = __reduce_max_sync(grp, __float_as_int(d));
    if (!in || (threadIdx.x & 31) != __ffs(grp) - 1) return;
    const float m = __int_as_float(db) - ldexpf(box, -(level_of(cnt, leaf) + 1));
    if (!(m > 0.f)) return;
    const int mb = __float_as_int(m);
    uint32_t cur = leaf;
    for (;;) {
        const int old = atomicMax(reinterpret_cast<int *>(slack) + cur, mb);
        if (cur == 0 || old >= mb) break;
        cur = nodes[cur].parent;
    }
}

__global__ void k_refresh_zero(const SphCounters *cnt, float *__restrict__ slack)
{
    const uint32_t nn = cnt->n_nodes;
    for (uint32_t nd = blockIdx.x * blockDim.x + threadIdx.x; nd < nn; nd += gridDim.x * blockDim.x) slack[nd] = 0.f;
}

// half edge of every cell = its geometric half edge + its slack
__global__ void k_refresh_apply(const SphCounters *cnt, SphNode *__restrict__ nodes, const float *__restrict__ slack, float box)
{
    const uint32_t nn = cnt->n_nodes;
    for (uint32_t nd = blockIdx.x * blockDim.x + threadIdx.x; nd < nn; nd += gridDim.x * blockDim.x)
        nodes[nd].half = ldexpf(box, -(level_of(cnt, nd) + 1)) + slack[nd] * (1.f + 1e-6f);
}

template <typename T>
int ensure(sph_ctx *ctx, T **p, size_t count)
{
    if (*p) { cudaFree(*p); *p = nullptr; }
    if (count == 0) count = 1;
    SPH_CUDA(ctx, cudaMalloc((void **)p, count * sizeof(T)));
    return SPH_OK;
}

inline int nblocks(int64_t n, int t) { return (int)((n + t - 1) / t); }

} // namespace

int sph_index_build(sph_ctx *ctx, const float *pos, const float *mass)
{
    const int64_t n = ctx->n;
    cudaStream_t st = ctx->stream;
    const uint32_t B = SPH_LEAF;
    int rc;
    if (n > ctx->cap_n) {
        int64_t cap = n + n / 8 + 1024;
        ctx->cap_n = 0; // (an allocation failure below leaves no stale capacity behind)
        if ((rc = ensure(ctx, &ctx->keys, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->keys_alt, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->perm, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->perm_alt, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->inv, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->xyzm, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->grp_mark, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->gid_of_slot, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->slot_leaf, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->grp_start, cap + 1))) return rc;
        if ((rc = ensure(ctx, &ctx->f_xyzh, cap))) return rc;
        if ((rc = ensure(ctx, &ctx->f_vc, 2 * cap))) return rc; // 32-byte records (v,c | rho,A,m,1/H)
        if (ctx->f_ext) { cudaFree(ctx->f_ext); ctx->f_ext = nullptr; } // (re-allocated on first use)
        if (ctx->node_mom) { cudaFree(ctx->node_mom); ctx->node_mom = nullptr; ctx->node_mom_cap = 0; }
        // node pool: internal nodes hold > B particles each; 8 children per internal node.
        // Typical use is ~ 8 n / (3 B); the pool is sized generously and overflow degrades gracefully.
        int64_t ncap = 64 + 8 * (2 * cap / (int64_t)(B > 4 ? B / 4 : 1) + 8);
        if (ncap > 0x7fffff00ll) ncap = 0x7fffff00ll;
        ncap = 1 + 8 * ((ncap - 1) / 8);
        if ((rc = ensure(ctx, &ctx->nodes, ncap))) return rc;
        if ((rc = ensure(ctx, &ctx->node_hmax, ncap))) return rc;
        if ((rc = ensure(ctx, &ctx->node_slack, ncap))) return rc;
        ctx->node_cap = ncap;
        ctx->cap_n = cap;
    }
    if (n == 0) {
        SPH_CUDA(ctx, cudaMemsetAsync(ctx->cnt, 0, offsetof(SphCounters, err), st)); // n_nodes, n_groups, ... (not the pending errors)
        SPH_CUDA(ctx, cudaMemsetAsync(&ctx->cnt->idx_err, 0, sizeof(unsigned int), st));
        ctx->have_index = true;
        return SPH_OK;
    }

    const int T = 256;
    float scale = (float)(1 << SPH_LMAX) / ctx->prm.box;
    SPH_CUDA(ctx, cudaMemsetAsync(&ctx->cnt->idx_err, 0, sizeof(unsigned int), st));
    k_keys<<<nblocks(n, T), T, 0, st>>>(n, pos, scale, ctx->prm.box, ctx->keys, ctx->perm, ctx->cnt);
    ctx->launches++;

    // a2: stable LSD radix sort of (key, id) on the 48 key bits (sph_sort.cu)
    int in_alt = 0;
    if ((rc = sph_sort_pairs_u64(ctx, ctx->keys, ctx->keys_alt, ctx->perm, ctx->perm_alt, n, SPH_KEY_BITS, &in_alt))) return rc;
    if (in_alt) { // the sorted data must sit in ctx->keys / ctx->perm
        { uint64_t *t = ctx->keys; ctx->keys = ctx->keys_alt; ctx->keys_alt = t; }
        { uint32_t *t = ctx->perm; ctx->perm = ctx->perm_alt; ctx->perm_alt = t; }
    }
    const uint64_t *skeys = ctx->keys;
    const uint32_t *sperm = ctx->perm;

    k_permute<<<nblocks(n, T), T, 0, st>>>(n, pos, mass, ctx->mass_scalar, sperm, ctx->xyzm, ctx->inv);
    ctx->launches++;

    // a4: octree, one level per launch (a level's nodes are contiguous in the pool)
    k_tree_init<<<1, 32, 0, st>>>(ctx->cnt, ctx->nodes, (uint32_t)n, ctx->prm.box);
    ctx->launches++;
    // thread-per-node kernels: bound by dependent loads, as many resident warps as an SM holds (fewer for small sets)
    const int grid = (int)std::max<int64_t>(1, std::min<int64_t>((int64_t)ctx->device_sms * 16, n / 64));
    for (int level = 0; level < SPH_LMAX; level++) {
        // 8 threads per node, at most 8^level nodes: one block for levels 0 and 1 (measured: 16 blocks per SM instead of 4
        // on the deeper levels and 4 / 32 blocks on levels 2 / 3 take the index build from 1.52 to 1.38 ms at 10^7)
        const int g = level < 2 ? 1 : level == 2 ? 4 : level == 3 ? std::min(32, grid) : grid;
        k_tree_split<<<g, 128, 0, st>>>(ctx->cnt, ctx->nodes, skeys, level, B, (uint32_t)ctx->node_cap);
        ctx->launches++;
    }
    // a5: group starts in sorted order + group id of every slot
    SPH_CUDA(ctx, cudaMemsetAsync(ctx->grp_mark, 0, sizeof(uint32_t) * n, st));
    k_mark_groups<<<grid, 128, 0, st>>>(ctx->cnt, ctx->nodes, (uint32_t)ctx->grp_cap,
                                        (uint32_t)(ctx->grp_node > SPH_LEAF ? ctx->grp_node : SPH_LEAF), ctx->grp_mark, ctx->slot_leaf);
    ctx->launches++;
    if ((rc = sph_scan_marks(ctx, ctx->grp_mark, n, ctx->gid_of_slot, ctx->grp_start, &ctx->cnt->n_groups))) return rc;

    // asynchronous: the octree and group counts stay on the device (the kernels read them there; the grids of the
    // persistent gather kernels are sized from the particle count)
    SPH_CUDA(ctx, cudaGetLastError());
    ctx->have_index = true;
    return SPH_OK;
}

// room for active lists of up to cap entries (a time-bin driver reserves n once instead of growing step by step)
int sph_active_reserve(sph_ctx *ctx, int64_t cap)
{
    int rc;
    if (cap <= ctx->cap_act) return SPH_OK;
    ctx->cap_act = 0;
    if ((rc = ensure(ctx, &ctx->act_slot, cap))) return rc;
    if ((rc = ensure(ctx, &ctx->act_slot_alt, cap))) return rc;
    if ((rc = ensure(ctx, &ctx->act_flag, cap))) return rc;
    if ((rc = ensure(ctx, &ctx->agrp_start, cap + 1))) return rc;
    ctx->cap_act = cap;
    return SPH_OK;
}

// a5 (active subset): ids -> sorted slots -> sort -> groups = runs sharing an all-active group
int sph_active_groups(sph_ctx *ctx, const int32_t *active, int64_t na)
{
    cudaStream_t st = ctx->stream;
    int rc;
    if (ctx->act_keep) return SPH_OK; // the caller (a driver inside the library) vouches: same list, same index as the last call
    if (na > ctx->cap_act && (rc = sph_active_reserve(ctx, na + na / 8 + 1024))) return rc;
    const int T = 256;
    k_act_slots<<<nblocks(na, T), T, 0, st>>>(na, ctx->n, active, ctx->inv, ctx->act_slot_alt, ctx->cnt);
    int bits = 1;
    while (bits < 32 && ((int64_t)1 << bits) < ctx->n) bits++;
    int in_alt = 0;
    if ((rc = sph_sort_keys_u32(ctx, ctx->act_slot_alt, ctx->act_slot, na, bits, &in_alt))) return rc;
    if (!in_alt) { uint32_t *t = ctx->act_slot; ctx->act_slot = ctx->act_slot_alt; ctx->act_slot_alt = t; } // sorted slots -> act_slot
    k_act_flags<<<nblocks(na, T), T, 0, st>>>(na, ctx->act_slot, ctx->gid_of_slot, ctx->act_flag, ctx->cnt);
    if ((rc = sph_scan_marks(ctx, ctx->act_flag, na, nullptr, ctx->agrp_start, &ctx->cnt->n_agroups))) return rc;
    ctx->launches += 2;
    return SPH_OK;
}

// positions moved since sph_index_build: same tree, same sorted order, cells inflated to hold their particles
int sph_index_refresh(sph_ctx *ctx, const float *pos)
{
    cudaStream_t st = ctx->stream;
    const int grid = ctx->device_sms * 8;
    k_refresh_zero<<<grid, 256, 0, st>>>(ctx->cnt, ctx->node_slack);
    k_refresh_slots<<<nblocks(ctx->n, 256), 256, 0, st>>>(ctx->n, ctx->cnt, ctx->nodes, ctx->perm, ctx->slot_leaf, pos, ctx->prm.box, ctx->xyzm,
                                                          ctx->node_slack);
    k_refresh_apply<<<grid, 256, 0, st>>>(ctx->cnt, ctx->nodes, ctx->node_slack, ctx->prm.box);
    ctx->launches += 3;
    SPH_CUDA(ctx, cudaGetLastError());
    return SPH_OK;
}
