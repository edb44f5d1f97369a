// sph_gather.cuh -- device code shared by the density and the force gather kernels (steps a5/a6):
// per-group octree walk that emits candidate leaf segments, staging of the segments' sorted float4
// runs into shared memory, and the split of a group's work into per-warp units.
//
// One CTA (4 warps) owns one group of <= 32 active particles that lie in one octree leaf -- the
// paper's "tree walk over groups of one or more active particles" (§1); candidates are
// processed 32 at a time per warp, the analogue of its N_chunk = 32 (PAPER.md:104 §2.4, :108 §3).
#pragma once

#include "sph_internal.cuh"

#define FULLMASK 0xffffffffu
// padding coordinate of lanes past the end of a candidate range: every comparison with NaN is
// false, in the plain and in the per-pair nearest-image frame alike
#define SPH_NANF __int_as_float(0x7fc00000)

// Minimum-image difference of two coordinates in [0, L) with the relative accuracy of a plain fp32
// difference: x - L is exact for x >= L/2 (Sterbenz), so the wrapped branch subtracts two nearby
// numbers instead of rounding the large difference first (which would leave an error of ulp(L) on a
// result that may be 1e-3 L).
__device__ __forceinline__ float image_diff(float xi, float cx, float L)
{
    float d = xi - cx;
    const float hl = 0.5f * L;
    if (d >= hl) d = (xi - L) - cx;
    else if (d < -hl) d = xi - (cx - L);
    return d;
}

__device__ __forceinline__ unsigned lanemask_lt()
{
    unsigned m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

__device__ __forceinline__ float warp_max(float v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fmaxf(v, __shfl_xor_sync(FULLMASK, v, o));
    return v;
}
__device__ __forceinline__ float warp_min(float v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v = fminf(v, __shfl_xor_sync(FULLMASK, v, o));
    return v;
}
__device__ __forceinline__ double warp_sum_d(double v)
{
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(FULLMASK, v, o);
    return v;
}

// Walk state kept in shared memory between batches of one evaluation.
struct WalkShared {
    uint32_t seg_start[SPH_SMAX];
    uint32_t seg_pre[SPH_SMAX + 1]; // exclusive prefix of segment lengths; [n_seg] = total
    uint32_t stack[SPH_STK];
    float gc[3], gh[3];   // group bounding box: centre, half extent (raw coordinates)
    float thr[3];         // zero-centred-frame threshold per axis (+inf: raw coordinates)
    float hg;             // group reach (max support radius of the unconverged actives)
    int sp;               // stack pointer (-1: walk not started)
    int n_seg;
    uint32_t total;       // candidates in this batch
    int pairwrap;         // 1: per-pair nearest image (reach comparable to the box)
};

__device__ __forceinline__ SphNode load_node(const SphNode *__restrict__ nodes, uint32_t i)
{
    const float4 *p = reinterpret_cast<const float4 *>(nodes + i);
    float4 a = __ldg(p), b = __ldg(p + 1);
    SphNode n;
    n.start = __float_as_uint(a.x); n.count = __float_as_uint(a.y);
    n.child = __float_as_uint(a.z); n.parent = __float_as_uint(a.w);
    n.cx = b.x; n.cy = b.y; n.cz = b.z; n.half = b.w;
    return n;
}

// Executed by warp 0.  Continues (or starts, ws.sp == -1) the depth-first walk and fills one batch of
// candidate segments: every leaf whose cell comes closer to the group's bounding box than the reach
// (density: hg; force: max(hg, largest support radius inside the node), the symmetric set of R10).
// Stack entries are blocks of 8 sibling nodes; each step pops up to 4 blocks (32 lanes, one node per
// lane) so that the stack holds at most 32 entries per tree level.
template <bool FORCE>
__device__ void walk_batch(WalkShared &ws, const SphNode *__restrict__ nodes, const float *__restrict__ node_hmax,
                           float L, uint32_t tile_cap, uint32_t n_nodes)
{
    const int lane = threadIdx.x & 31;
    int sp = ws.sp, n_seg = 0;
    uint32_t total_est = 0;
    float maxhalf = 0.f, maxreach = ws.hg;
    const float gcx = ws.gc[0], gcy = ws.gc[1], gcz = ws.gc[2];
    const float ghx = ws.gh[0], ghy = ws.gh[1], ghz = ws.gh[2];
    const float pad = 1e-6f * L;
    if (sp < 0) { // start
        SphNode root = load_node(nodes, 0);
        sp = 0;
        if (root.child == 0) {
            if (root.count > 0 && lane == 0) { ws.seg_start[0] = root.start; ws.seg_pre[0] = root.count; }
            if (root.count > 0) { n_seg = 1; maxhalf = root.half; total_est = root.count; }
            if (FORCE) maxreach = fmaxf(maxreach, __ldg(node_hmax));
        } else {
            if (lane == 0) ws.stack[0] = root.child;
            sp = 1;
        }
        __syncwarp();
    }
    // stop a batch once it holds a few tiles worth of candidates (bounds smem lists, keeps tiles full)
    while (sp > 0 && n_seg <= SPH_SMAX - 32 && total_est < 4u * tile_cap) {
        int npop = min(sp, 4);
        sp -= npop;
        int e = lane >> 3;
        bool valid = e < npop;
        uint32_t idx = valid ? ws.stack[sp + e] + (lane & 7) : 0u;
        SPH_ASSERT(sp + 4 <= SPH_STK && idx < n_nodes);
        SphNode nd = load_node(nodes, idx);
        float reach = ws.hg;
        if (FORCE) reach = fmaxf(reach, __ldg(node_hmax + idx));
        float hh = nd.half * (1.f + 1e-6f) + pad;
        float dx = fabsf(gcx - nd.cx); dx = fminf(dx, L - dx); dx = fmaxf(dx - (ghx + hh), 0.f);
        float dy = fabsf(gcy - nd.cy); dy = fminf(dy, L - dy); dy = fmaxf(dy - (ghy + hh), 0.f);
        float dz = fabsf(gcz - nd.cz); dz = fminf(dz, L - dz); dz = fmaxf(dz - (ghz + hh), 0.f);
        float d2 = dx * dx + dy * dy + dz * dz;
        float rp = reach * (1.f + 1e-5f);
        bool pass = valid && nd.count > 0 && d2 <= rp * rp;
        bool leaf = nd.child == 0;
        bool emit = pass && leaf, push = pass && !leaf;
        unsigned me = __ballot_sync(FULLMASK, emit);
        if (emit) {
            int p = n_seg + __popc(me & lanemask_lt());
            SPH_ASSERT(p < SPH_SMAX);
            ws.seg_start[p] = nd.start;
            ws.seg_pre[p] = nd.count;
            maxhalf = fmaxf(maxhalf, nd.half);
            maxreach = fmaxf(maxreach, reach);
        }
        n_seg += __popc(me);
        uint32_t c = emit ? nd.count : 0u;
#pragma unroll
        for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(FULLMASK, c, o);
        total_est += c;
        unsigned mp = __ballot_sync(FULLMASK, push);
        SPH_ASSERT(sp + __popc(mp) <= SPH_STK);
        if (push) ws.stack[sp + __popc(mp & lanemask_lt())] = nd.child;
        sp += __popc(mp);
        __syncwarp();
    }
    maxhalf = warp_max(maxhalf);
    maxreach = warp_max(maxreach);
    __syncwarp();
    // exclusive prefix of the segment lengths (in place)
    uint32_t carry = 0;
    for (int b = 0; b < n_seg; b += 32) {
        int i = b + lane;
        uint32_t v = i < n_seg ? ws.seg_pre[i] : 0u, inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t t = __shfl_up_sync(FULLMASK, inc, o);
            if (lane >= o) inc += t;
        }
        if (i < n_seg) ws.seg_pre[i] = carry + inc - v;
        carry += __shfl_sync(FULLMASK, inc, 31);
    }
    if (lane == 0) {
        ws.seg_pre[n_seg] = carry;
        ws.sp = sp;
        ws.n_seg = n_seg;
        ws.total = carry;
        // Frame choice.  If everything involved lies within L/4 of the group centre, coordinates of the
        // actives and of the candidates are brought into one frame in which plain differences ARE the
        // minimum-image differences: raw coordinates when the group sits in the middle half of the axis,
        // else the zero-centred frame x -> x - L for x >= L/2 (exact in fp32, Sterbenz).  Otherwise
        // (reach comparable to the box) fall back to a per-pair nearest image.
        float ext = fmaxf(ghx, fmaxf(ghy, ghz)) + maxreach * (1.f + 1e-5f) + 2.f * maxhalf + 4.f * pad;
        int pw = !(ext < 0.25f * L);
        ws.pairwrap = pw;
        const float inf = __int_as_float(0x7f800000);
        ws.thr[0] = (pw || (gcx >= 0.25f * L && gcx < 0.75f * L)) ? inf : 0.5f * L;
        ws.thr[1] = (pw || (gcy >= 0.25f * L && gcy < 0.75f * L)) ? inf : 0.5f * L;
        ws.thr[2] = (pw || (gcz >= 0.25f * L && gcz < 0.75f * L)) ? inf : 0.5f * L;
    }
}

// Copy the part of the batch's flat candidate range [tile_base, tile_base + tile_cap) into shared
// memory, one warp per segment (a segment is a contiguous, 16-byte aligned run of the sorted float4
// arrays), applying the frame shift to the coordinates.
template <int NARR>
__device__ __forceinline__ void stage_tile(const WalkShared &ws, float4 *const *tiles /*NARR smem arrays*/,
                                           const float4 *const *src /*NARR global arrays*/, uint32_t tile_base,
                                           uint32_t tile_cap, float L)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t t_lo = tile_base, t_hi = min(tile_base + tile_cap, ws.total);
    const float tx = ws.thr[0], ty = ws.thr[1], tz = ws.thr[2];
    for (int s = warp; s < ws.n_seg; s += SPH_WARPS) {
        uint32_t p0 = ws.seg_pre[s], p1 = ws.seg_pre[s + 1];
        if (p1 <= t_lo || p0 >= t_hi) continue;
        uint32_t lo = max(p0, t_lo), hi = min(p1, t_hi);
        uint32_t gsrc = ws.seg_start[s] - p0;
        for (uint32_t e = lo + lane; e < hi; e += 32) {
            SPH_ASSERT(e - t_lo < tile_cap);
            const uint32_t gi = gsrc + e; // modulo 2^32: seg_start - p0 may wrap
            float4 v = __ldg(src[0] + gi);
            v.x -= (v.x >= tx) ? L : 0.f;
            v.y -= (v.y >= ty) ? L : 0.f;
            v.z -= (v.z >= tz) ? L : 0.f;
            tiles[0][e - t_lo] = v;
#pragma unroll
            for (int a = 1; a < NARR; a++) tiles[a][e - t_lo] = __ldg(src[a] + gi);
        }
    }
}

// Split of n_u actives x tn candidates into units for the 4 warps: blocks of <= 4 actives
// (register-blocked), and for fewer than 4 actives also parts of the candidate range.
struct UnitPlan {
    int nb, parts;
};
__device__ __forceinline__ UnitPlan plan_units(int n_u)
{
    UnitPlan p;
    if (n_u >= SPH_WARPS) {
        p.nb = (((n_u + SPH_ABLK - 1) / SPH_ABLK) + SPH_WARPS - 1) & ~(SPH_WARPS - 1);
        p.parts = 1;
    } else {
        p.nb = n_u;
        p.parts = n_u > 0 ? SPH_WARPS / n_u : 1;
    }
    return p;
}
