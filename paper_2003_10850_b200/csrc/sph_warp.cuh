// sph_warp.cuh -- device code shared by the gather kernels (steps a5/a6): the octree walk that emits
// the candidate set of a group as runs of the sorted order, and the shared-memory primitives.
//
// One CTA owns one group of <= 32 active particles that are consecutive in the sorted order inside one
// small octree node -- the paper's "tree walk over groups of one or more active particles"
// (§1).  Warp 0 of the CTA walks the tree for the whole group; all warps then stage the
// candidate runs in shared memory and test them (sph_density.cu, sph_force.cu).  The staged tile plays
// the role of the paper's N_chunk (PAPER.md:104 §2.4, :108 §3): candidates are consumed tile by tile,
// never as per-particle neighbour lists in memory.
#pragma once

#include "sph_internal.cuh"

#define FULLMASK 0xffffffffu
#define SPH_NANF __int_as_float(0x7fc00000)

// Minimum-image difference of two coordinates in [0, L) with the relative accuracy of a plain fp32
// difference: x - L is exact for x >= L/2 (Sterbenz), so the wrapped branch subtracts two nearby
// numbers instead of rounding the large difference first.
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

// ---------------------------------------------------------------------------------------------
// shared-memory primitives
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// Hit-queue stores.  The queue of a lane is written and read by that lane only, through these asm
// statements and the (volatile, memory-clobbering) queue loads of the drain loops, which stay ordered
// after them; leaving the clobber off here lets the compiler hoist the next candidates' shared-memory
// loads above the pushes of the previous test, so that the unrolled tests overlap.
__device__ __forceinline__ void sts_f32(uint32_t addr, float v)
{
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v)); // no memory clobber: see hit-queue note
}
__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v));
}

__device__ __forceinline__ uint32_t lds_u32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}

// ---------------------------------------------------------------------------------------------
// Walk state of a group, in shared memory.
struct WalkShared {
    uint32_t seg_start[SPH_SMAX];   // first sorted slot of each candidate segment (a run of the sorted order)
    uint32_t seg_pre[SPH_SMAX + 1]; // exclusive prefix of the segment lengths; [n_seg] = total
    uint32_t stack[SPH_STK];        // blocks of 8 sibling nodes still to visit
    int sp, n_seg;                  // stack pointer and segment count between the steps of a batch
    int wcnt[SPH_WARPS][2];         // per warp: segment heads / pushes of the current step
    float wmax[SPH_WARPS][2];       // per warp: largest emitted cell half edge, largest reach
    float box[7];                   // the group: bounding box centre (3), half extent (3), reach
    // Result of the batch.  Frame (see the end of walk_cta): per axis, coordinates >= thr are shifted
    // by -L (thr = +inf: axis untouched); pairwrap: per-pair nearest image needed instead.
    uint32_t total;
    float thx, thy, thz;
    int pairwrap;
};

// the batch result as registers of every thread
struct WalkCtl {
    int sp, n_seg;
    uint32_t total;
    float thx, thy, thz;
    bool pairwrap;
};
__device__ __forceinline__ WalkCtl walk_result(const WalkShared &W)
{
    WalkCtl c;
    c.sp = W.sp; c.n_seg = W.n_seg; c.total = W.total;
    c.thx = W.thx; c.thy = W.thy; c.thz = W.thz; c.pairwrap = W.pairwrap != 0;
    return c;
}

// coordinate in the batch's frame: exact (x - L is exact for x >= L/2, Sterbenz)
__device__ __forceinline__ float recentre(float x, float thr, float L) { return x >= thr ? x - L : x; }

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

// Starts (start = true) or continues the depth-first walk of the CTA's group and fills one batch of
// candidate segments: every leaf whose cell comes closer to the group's bounding box (W.box: centre,
// half extent) than the reach (density: hg = W.box[6]; force: max(hg, largest support radius inside
// the node), the symmetric set of R10), and every cell that lies wholly within hg of the box.  Called
// by ALL threads of the CTA: a step pops up to 16 blocks of 8 siblings, one node per thread, so the
// chain of dependent node loads is as short as the tree is deep, not as long as the candidate list.
// Stack bound: 16-block pops only while sp <= SPH_STK16 (+112 at most), single-block pops grow the
// stack by <= 7 per tree level: sp <= SPH_STK16 + 112 + 8 * SPH_LMAX <= SPH_STK.
// On return (after a __syncthreads) W.sp > 0 means the walk is not finished: call again.
template <bool FORCE>
__device__ __forceinline__ void walk_cta(WalkShared &W, const SphNode *__restrict__ nodes,
                                         const float *__restrict__ node_hmax, float L, bool start)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float gcx = W.box[0], gcy = W.box[1], gcz = W.box[2], ghx = W.box[3], ghy = W.box[4], ghz = W.box[5];
    const float hg = W.box[6];
    float maxhalf = 0.f, maxreach = hg;
    const float pad = 1e-6f * L;
    if (tid == 0) {
        W.n_seg = 0;
        if (start) {
            SphNode root = load_node(nodes, 0);
            W.sp = 0;
            if (root.child == 0) {
                if (root.count > 0) {
                    W.seg_start[0] = root.start; W.seg_pre[0] = root.count;
                    W.n_seg = 1; maxhalf = root.half;
                }
                if (FORCE) maxreach = fmaxf(maxreach, __ldg(node_hmax));
            } else {
                W.stack[0] = root.child;
                W.sp = 1;
            }
        }
    }
    for (;;) {
        __syncthreads();
        const int sp0 = W.sp, ns0 = W.n_seg;
        if (sp0 <= 0 || ns0 > SPH_SMAX - SPH_THREADS) break;
        const int npop = sp0 <= SPH_STK16 ? min(sp0, SPH_THREADS / 8) : 1;
        const int e = tid >> 3;
        const bool valid = e < npop;
        const uint32_t idx = valid ? W.stack[sp0 - npop + e] + (tid & 7) : 0u;
        SphNode nd = load_node(nodes, idx);
        float reach = hg;
        if (FORCE) reach = fmaxf(reach, __ldg(node_hmax + idx));
        const float hh = nd.half * (1.f + 1e-6f) + pad;
        const float ax = fabsf(gcx - nd.cx), ay = fabsf(gcy - nd.cy), az = fabsf(gcz - nd.cz);
        const float mx = fminf(ax, L - ax), my = fminf(ay, L - ay), mz = fminf(az, L - az); // periodic separation of the centres
        const float dx = fmaxf(mx - (ghx + hh), 0.f), dy = fmaxf(my - (ghy + hh), 0.f), dz = fmaxf(mz - (ghz + hh), 0.f);
        const float d2 = dx * dx + dy * dy + dz * dz;
        const float rp = reach * (1.f + 1e-5f);
        const bool pass = valid && nd.count > 0 && d2 <= rp * rp;
        const bool leaf = nd.child == 0;
        // A cell EVERY point of which lies within the group's own reach of the bounding box is emitted
        // whole, as one long run of the sorted order: none of its descendants could be pruned (their
        // nearest point is no farther than that), so descending would only cut the run into pieces.
        const float fx = fmaxf(mx + hh - ghx, 0.f), fy = fmaxf(my + hh - ghy, 0.f), fz = fmaxf(mz + hh - ghz, 0.f);
        const bool inside = fx * fx + fy * fy + fz * fz <= hg * hg;
        const bool emit = pass && (leaf || inside), push = pass && !emit;
        // Sibling cells are consecutive runs of the sorted order: a run of emitted siblings (empty ones
        // in between do not matter) becomes ONE segment, emitted by the run's first lane.
        const unsigned me = __ballot_sync(FULLMASK, emit);
        const unsigned mbrk = __ballot_sync(FULLMASK, valid && nd.count > 0 && !emit);
        const unsigned blk = 0xffu << (lane & 24);                 // the 8 lanes of this lane's sibling block
        const unsigned below = blk & lanemask_lt(), above = blk & ~lanemask_lt() & ~(1u << lane);
        const unsigned prevs = (me | mbrk) & below;                 // non-empty siblings before this one
        const bool head = emit && (prevs == 0u || ((mbrk >> (31 - __clz(prevs))) & 1u));
        const unsigned nb = mbrk & above;                           // first break after this lane ends the run
        const unsigned runm = me & (above | (1u << lane)) & (nb ? ((1u << (__ffs(nb) - 1)) - 1u) : 0xffffffffu);
        const int last = 31 - __clz(runm | (1u << lane));           // last emitted sibling of the run
        const uint32_t endpos = __shfl_sync(FULLMASK, nd.start + nd.count, last);
        const unsigned mh = __ballot_sync(FULLMASK, head);
        const unsigned mp = __ballot_sync(FULLMASK, push);
        if (emit) {
            if (!inside) maxhalf = fmaxf(maxhalf, nd.half); // (every point of an inside cell lies within hg of the box)
            maxreach = fmaxf(maxreach, reach);
        }
        if (lane == 0) { W.wcnt[warp][0] = __popc(mh); W.wcnt[warp][1] = __popc(mp); }
        __syncthreads();
        int sb = ns0, pb = sp0 - npop, st = 0, pt = 0;
#pragma unroll
        for (int w = 0; w < SPH_WARPS; w++) {
            const int a = W.wcnt[w][0], b = W.wcnt[w][1];
            if (w < warp) { sb += a; pb += b; }
            st += a; pt += b;
        }
        if (head) {
            const int p = sb + __popc(mh & lanemask_lt());
            SPH_ASSERT(p < SPH_SMAX);
            W.seg_start[p] = nd.start;
            W.seg_pre[p] = endpos - nd.start;
        }
        if (push) {
            SPH_ASSERT(pb + __popc(mp & lanemask_lt()) < SPH_STK);
            W.stack[pb + __popc(mp & lanemask_lt())] = nd.child;
        }
        if (tid == 0) { W.sp = sp0 - npop + pt; W.n_seg = ns0 + st; }
    }
    // (every thread has passed the loop's last barrier; W.sp / W.n_seg are final)
    maxhalf = warp_max(maxhalf);
    maxreach = warp_max(maxreach);
    if (lane == 0) { W.wmax[warp][0] = maxhalf; W.wmax[warp][1] = maxreach; }
    const int n_seg = W.n_seg;
    if (warp == 0) {
        // exclusive prefix of the segment lengths (in place)
        uint32_t carry = 0;
        for (int b = 0; b < n_seg; b += 32) {
            const int i = b + lane;
            const uint32_t v = i < n_seg ? W.seg_pre[i] : 0u;
            uint32_t inc = v;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t t = __shfl_up_sync(FULLMASK, inc, o);
                if (lane >= o) inc += t;
            }
            if (i < n_seg) W.seg_pre[i] = carry + inc - v;
            carry += __shfl_sync(FULLMASK, inc, 31);
        }
        if (lane == 0) { W.seg_pre[n_seg] = carry; W.total = carry; }
    }
    __syncthreads();
    if (tid == 0) {
#pragma unroll
        for (int w = 0; w < SPH_WARPS; w++) { maxhalf = fmaxf(maxhalf, W.wmax[w][0]); maxreach = fmaxf(maxreach, W.wmax[w][1]); }
        // Frame choice, per axis.  ext bounds how far any candidate of this batch can lie from the group's
        // bounding box.  (i) The group, its reach and every candidate cell stay clear of both box faces:
        // plain differences of raw coordinates ARE the minimum-image differences (thr = +inf).  (ii) They
        // cross a face but span less than half the box: map every coordinate x >= L/2 to x - L (exact), for
        // actives and candidates alike; all of them then lie in one interval inside (-L/2, L/2) and plain
        // differences are again the minimum-image differences, while a candidate outside that span can only
        // look farther away than it is, never closer.  (iii) Otherwise (a reach comparable to the box):
        // per-pair image.
        const float inf = __int_as_float(0x7f800000);
        const float ext = maxreach * (1.f + 1e-5f) + 2.f * maxhalf + 4.f * pad;
        const float hl = 0.5f * L, ql = 0.249f * L; // span = 2 (gh + ext) < L/2
        const bool okx = gcx - ghx - ext >= 0.f && gcx + ghx + ext < L;
        const bool oky = gcy - ghy - ext >= 0.f && gcy + ghy + ext < L;
        const bool okz = gcz - ghz - ext >= 0.f && gcz + ghz + ext < L;
        W.thx = okx ? inf : hl;
        W.thy = oky ? inf : hl;
        W.thz = okz ? inf : hl;
        W.pairwrap = ((!okx && ghx + ext >= ql) || (!oky && ghy + ext >= ql) || (!okz && ghz + ext >= ql)) ? 1 : 0;
    }
    __syncthreads();
}

// the group's bounding box and reach, published by warp 0 (has: this lane holds an active of the group)
__device__ __forceinline__ void publish_box(WalkShared &W, bool has, float x, float y, float z, float reach)
{
    const float inf = __int_as_float(0x7f800000);
    const float x0 = warp_min(has ? x : inf), x1 = warp_max(has ? x : -inf);
    const float y0 = warp_min(has ? y : inf), y1 = warp_max(has ? y : -inf);
    const float z0 = warp_min(has ? z : inf), z1 = warp_max(has ? z : -inf);
    if ((threadIdx.x & 31) == 0) {
        W.box[0] = 0.5f * (x0 + x1); W.box[3] = 0.5f * (x1 - x0) * (1.f + 1e-6f);
        W.box[1] = 0.5f * (y0 + y1); W.box[4] = 0.5f * (y1 - y0) * (1.f + 1e-6f);
        W.box[2] = 0.5f * (z0 + z1); W.box[5] = 0.5f * (z1 - z0) * (1.f + 1e-6f);
        W.box[6] = reach;
    }
}

__device__ __forceinline__ float4 ldg_nc(const float4 *p)
{
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// segment that holds flat position p: largest k < n_seg with seg_pre[k] <= p (branch-free bisection)
__device__ __forceinline__ int seg_of(const WalkShared &W, int n_seg, uint32_t p)
{
    int k = 0;
#pragma unroll
    for (int step = SPH_SMAX / 2; step; step >>= 1) {
        const int k2 = k + step;
        if (k2 < n_seg && W.seg_pre[k2] <= p) k = k2;
    }
    return k;
}

// Thread layout of a group of g actives in a CTA: thread = a + g * s with a < g the active and s < f the
// candidate stream, f = floor(SPH_THREADS / g); stream s tests the candidate quads s, s + f, s + 2f, ...
__device__ __forceinline__ int streams_for(int g) { return SPH_THREADS / g; }

// ---------------------------------------------------------------------------------------------
// Order in which a staged set of cnt candidates is consumed.  The walk emits candidates in Morton
// (depth-first) order, so consecutive flat positions are spatial neighbours: they are inside or outside
// an active's support TOGETHER.  Tested in that order, (i) at any time only the threads whose active
// lies near the current stretch collect hits, and (ii) a thread's share of the hits, taken in clumps,
// scatters by a factor of two around the mean -- either way the bulk evaluation of queued hits runs on
// a few lanes.  The set is therefore dealt candidate by candidate, round-robin, onto SPH_PILES piles
// that are stored one after the other (slot = (o mod P) * pl + o / P): every stretch of the stored
// order is a uniform sample of the whole set and no two candidates of a quad are neighbours, so every
// thread meets its hits at a steady rate and ends with its fair share.  pl is odd: the 32 lanes of a
// gather window store into 32 different piles, i.e. 32 different banks.
#define SPH_PILES 64
struct PileMap {
    uint32_t pl;   // slots per pile
    uint32_t np;   // slots in use = SPH_PILES * pl (a multiple of 64)
};
__device__ __forceinline__ PileMap pile_map(uint32_t cnt)
{
    PileMap m;
    m.pl = ((cnt + SPH_PILES - 1u) / SPH_PILES) | 1u;
    m.np = SPH_PILES * m.pl;
    return m;
}
__device__ __forceinline__ uint32_t pile_slot(const PileMap &m, uint32_t o) // flat offset in the set -> stored slot
{
    return (o & (SPH_PILES - 1u)) * m.pl + o / SPH_PILES;
}
#define SPH_PILE_SLACK (2 * SPH_PILES) // slots a set of cnt candidates can need beyond cnt (rounding of pl)
