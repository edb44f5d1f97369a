// sph_warp.cuh -- device code shared by the warp-per-group gather kernels (steps a5/a6):
// per-warp octree walk that emits candidate leaf segments, and the cooperative gather that stages a
// chunk of candidates in the warp's shared-memory slot as pair records for packed f32x2 tests.
//
// One WARP owns one group of <= 32 active particles that are consecutive in the sorted order inside
// one octree leaf -- the paper's "tree walk over groups of one or more active particles"
// (§1).  Warps never synchronise with one another: walk latency of one group hides
// behind the pair arithmetic of the others.  The chunk plays the role of the paper's N_chunk
// (PAPER.md:104 §2.4, :108 §3): candidates are consumed in fixed-size chunks, not as whole lists.
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
// Per-warp walk state.
struct WarpWalk {
    uint32_t seg_start[SPH_SMAX];   // first sorted slot of each candidate segment (a leaf)
    uint32_t seg_pre[SPH_SMAX + 1]; // exclusive prefix of the segment lengths; [n_seg] = total
    uint32_t stack[SPH_STK];        // blocks of 8 sibling nodes still to visit
};

struct WalkCtl { // warp-uniform registers
    int sp;        // stack pointer; -1: walk not started
    int n_seg;
    uint32_t total;
    // Frame of this batch (see the end of walk_batch): per axis, coordinates >= thr are shifted by -L
    // (thr = +inf: axis untouched); pairwrap: per-pair nearest image needed instead.
    float thx, thy, thz;
    bool pairwrap;
};

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

// Continues (or starts, ctl.sp == -1) the depth-first walk of this warp's group and fills one batch
// of candidate segments: every leaf whose cell comes closer to the group's bounding box (centre gc,
// half extent gh) than the reach (density: hg; force: max(hg, largest support radius inside the
// node), the symmetric set of R10).  Stack entries are blocks of 8 siblings; a step pops up to 4
// blocks (one node per lane).  Stack bound: 4-block pops only while sp <= SPH_STK4, single-block
// pops grow the stack by <= 7 per tree level, so sp <= SPH_STK4 + 28 + 7 * SPH_LMAX < SPH_STK.
template <bool FORCE>
__device__ __forceinline__ void walk_batch(WarpWalk &ws, WalkCtl &ctl, const SphNode *__restrict__ nodes,
                                           const float *__restrict__ node_hmax, float L, float gcx, float gcy,
                                           float gcz, float ghx, float ghy, float ghz, float hg)
{
    const int lane = threadIdx.x & 31;
    int sp = ctl.sp, n_seg = 0;
    float maxhalf = 0.f, maxreach = hg;
    const float pad = 1e-6f * L;
    __syncwarp();
    if (sp < 0) { // start
        SphNode root = load_node(nodes, 0);
        sp = 0;
        if (root.child == 0) {
            if (root.count > 0) {
                if (lane == 0) { ws.seg_start[0] = root.start; ws.seg_pre[0] = root.count; }
                n_seg = 1; maxhalf = root.half;
            }
            if (FORCE) maxreach = fmaxf(maxreach, __ldg(node_hmax));
        } else {
            if (lane == 0) ws.stack[0] = root.child;
            sp = 1;
        }
        __syncwarp();
    }
    while (sp > 0 && n_seg <= SPH_SMAX - 32) {
        int npop = sp <= SPH_STK4 ? min(sp, 4) : 1;
        sp -= npop;
        int e = lane >> 3;
        bool valid = e < npop;
        uint32_t idx = valid ? ws.stack[sp + e] + (lane & 7) : 0u;
        SphNode nd = load_node(nodes, idx);
        float reach = hg;
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
        // Sibling leaves are consecutive runs of the sorted order: a run of emitted siblings (empty ones
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
        if (emit) {
            maxhalf = fmaxf(maxhalf, nd.half);
            maxreach = fmaxf(maxreach, reach);
        }
        if (head) {
            int p = n_seg + __popc(mh & lanemask_lt());
            SPH_ASSERT(p < SPH_SMAX);
            ws.seg_start[p] = nd.start;
            ws.seg_pre[p] = endpos - nd.start;
        }
        n_seg += __popc(mh);
        unsigned mp = __ballot_sync(FULLMASK, push);
        SPH_ASSERT(sp + __popc(mp) <= SPH_STK);
        if (push) ws.stack[sp + __popc(mp & lanemask_lt())] = nd.child;
        sp += __popc(mp);
        __syncwarp();
    }
    maxhalf = warp_max(maxhalf);
    maxreach = warp_max(maxreach);
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
    if (lane == 0) ws.seg_pre[n_seg] = carry;
    __syncwarp();
    ctl.sp = sp;
    ctl.n_seg = n_seg;
    ctl.total = carry;
    // Frame choice, per axis.  ext bounds how far any candidate of this batch can lie from the group's
    // bounding box.  (i) The group, its reach and every candidate cell stay clear of both box faces:
    // plain differences of raw coordinates ARE the minimum-image differences (thr = +inf).  (ii) They
    // cross a face but span less than half the box: map every coordinate x >= L/2 to x - L (exact), for
    // actives and candidates alike; all of them then lie in one interval inside (-L/2, L/2) and plain differences are
    // again the minimum-image differences, while a candidate outside that span can only look farther
    // away than it is, never closer.  (iii) Otherwise (a reach comparable to the box): per-pair image.
    const float inf = __int_as_float(0x7f800000);
    const float ext = maxreach * (1.f + 1e-5f) + 2.f * maxhalf + 4.f * pad;
    const float hl = 0.5f * L, ql = 0.249f * L; // span = 2 (gh + ext) < L/2
    const bool okx = gcx - ghx - ext >= 0.f && gcx + ghx + ext < L;
    const bool oky = gcy - ghy - ext >= 0.f && gcy + ghy + ext < L;
    const bool okz = gcz - ghz - ext >= 0.f && gcz + ghz + ext < L;
    ctl.thx = okx ? inf : hl;
    ctl.thy = oky ? inf : hl;
    ctl.thz = okz ? inf : hl;
    ctl.pairwrap = (!okx && ghx + ext >= ql) || (!oky && ghy + ext >= ql) || (!okz && ghz + ext >= ql);
}

// ---------------------------------------------------------------------------------------------
// Candidate staging.  A batch's candidates form one flat index space [0, total) (segment k covers
// [seg_pre[k], seg_pre[k+1])); chunk c = flat range [c*CH, c*CH+CH).  The warp gathers a chunk into its
// shared-memory slot itself: lane l takes the four consecutive entries 4l..4l+3, finds their segments
// (segment heads become bits of a warp-uniform mask; the rank of a position is a population count), loads the
// four float4 records (one 64-byte run per lane unless a segment boundary intervenes), moves the
// coordinates into the batch's frame (recentre) and writes them as PAIR records, pair p of the chunk =
//   slot[p] = (x0,x1,y0,y1)   slot[SPH_CH/2 + p] = (z0,z1,w0,w1)
// so that the test loops load register pairs ready for packed f32x2 arithmetic.  Entries beyond the
// ragged tail become NaN (every comparison with NaN is false).
//
// Why not TMA bulk copies here (they were the first design, profiles/r1c_packed_tma.md): octree leaves hold ~8
// particles on average, so a chunk is ~10 pieces of ~100 bytes at arbitrary 16-byte offsets; every
// piece is one UBLKCP issued through uniform registers, which the compiler serialises lane by lane
// (ELECT / R2UR / UBLKCP, ~10 issue slots and a long-scoreboard wait per piece): 30 % of the kernel's
// time went there.  Tiles this small and irregular are not TMA's case; per-lane 16-byte loads are.
struct GatherCtl { // warp-uniform registers
    int kseg; // first segment that overlaps the next chunk to gather
};

// MUFU.RSQ / MUFU.RCP without the denormal scaling the C intrinsics wrap around them (arguments here are normal numbers:
// r^2 clamped to >= 1e-37, a sum of two densities); for normal arguments the results are those of rsqrtf / __fdividef(1, x)
__device__ __forceinline__ float rsqrt_ftz(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float sqrt_ftz(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float ex2_ftz(float x) // 2^x, MUFU.EX2 without the range wrapper of __expf (|x| small here)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_ftz(float x)
{
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float4 ldg_nc(const float4 *p)
{
    float4 v;
    asm volatile("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// The gather is split in two, so that the loads of chunk c + 1 can be in flight while chunk c is
// tested: gather_load computes the addresses and issues the 16-byte loads into registers, gather_store
// (after the consumer is done with the slot) fixes up and writes the pair records
// (slotp: [SPH_CH] float4; gidx: [SPH_CH] sorted slot of every entry or NULL).
struct GatherRegs {
    float4 c[4];   // entries 2 l, 2 l + 1, 2 (l + 32), 2 (l + 32) + 1 of the chunk
    uint32_t j[4]; // their sorted slots
    uint32_t lo, hi;
};

__device__ __forceinline__ void gather_load(const WarpWalk &ws, const WalkCtl &ctl, GatherCtl &gc, uint32_t chunk,
                                            GatherRegs &G, const float4 *__restrict__ src)
{
    const int lane = threadIdx.x & 31;
    const uint32_t lo = chunk * SPH_CH, hi = min(lo + SPH_CH, ctl.total);
    G.lo = lo; G.hi = hi;
    const int kfirst = gc.kseg;
    uint32_t w0 = 0u, w1 = 0u, w2 = 0u, w3 = 0u;
    int k0 = kfirst;
    for (;;) {
        const int k = k0 + lane;
        const bool in = k < ctl.n_seg;
        const uint32_t p0 = in ? ws.seg_pre[k] : 0xffffffffu, p1 = in ? ws.seg_pre[k + 1] : 0xffffffffu;
        const bool ov = in && p0 < hi && p1 > lo;
        const uint32_t pos = max(p0, lo) - lo, bit = ov ? 1u << (pos & 31u) : 0u, wd = pos >> 5;
        w0 |= __reduce_or_sync(FULLMASK, wd == 0u ? bit : 0u);
        w1 |= __reduce_or_sync(FULLMASK, wd == 1u ? bit : 0u);
        w2 |= __reduce_or_sync(FULLMASK, wd == 2u ? bit : 0u);
        w3 |= __reduce_or_sync(FULLMASK, wd == 3u ? bit : 0u);
        const unsigned m = __ballot_sync(FULLMASK, in && p1 > hi);
        if (m) { k0 += __ffs(m) - 1; break; }
        k0 += 32;
        if (k0 >= ctl.n_seg) { k0 = ctl.n_seg; break; }
    }
    gc.kseg = k0;
#pragma unroll
    for (int r = 0; r < 2; r++) {
        const int pr = lane + 32 * r;
        if (pr < SPH_CH / 2) {
            const int e0 = 2 * pr, wl = e0 >> 5, sh = e0 & 31;
            const uint32_t wmine = wl == 0 ? w0 : wl == 1 ? w1 : wl == 2 ? w2 : w3;
            const int below = kfirst - 1 + (wl > 0 ? __popc(w0) : 0) + (wl > 1 ? __popc(w1) : 0) + (wl > 2 ? __popc(w2) : 0);
            const int ka = below + __popc(wmine & (0xffffffffu >> (31 - sh)));
            const int kb = below + __popc(wmine & (0xffffffffu >> (30 - sh)));
            SPH_ASSERT(ka >= kfirst && kb < ctl.n_seg);
            const uint32_t pa = min(lo + e0, hi - 1u), pb = min(lo + e0 + 1u, hi - 1u);
            G.j[2 * r] = ws.seg_start[ka] + (pa - ws.seg_pre[ka]);
            G.j[2 * r + 1] = ws.seg_start[kb] + (pb - ws.seg_pre[kb]);
            G.c[2 * r] = ldg_nc(src + G.j[2 * r]);
            G.c[2 * r + 1] = ldg_nc(src + G.j[2 * r + 1]);
        }
    }
}

template <bool SQUARE_W, bool NEED_W>
__device__ __forceinline__ void gather_store(const WalkCtl &ctl, GatherRegs &G, float4 *slotp, uint32_t *gidx, float L)
{
    const int lane = threadIdx.x & 31;
    __syncwarp(); // every lane is done reading the slot's previous contents
    const bool rec = !ctl.pairwrap && (ctl.thx < 1e30f || ctl.thy < 1e30f || ctl.thz < 1e30f); // warp-uniform
#pragma unroll
    for (int r = 0; r < 2; r++) {
        const int pr = lane + 32 * r;
        if (pr < SPH_CH / 2) {
            float4 ca = G.c[2 * r], cb = G.c[2 * r + 1];
            const uint32_t e0 = 2u * pr;
            if (G.lo + e0 >= G.hi) ca.x = SPH_NANF;
            if (G.lo + e0 + 1u >= G.hi) cb.x = SPH_NANF;
            if (rec) {
                ca.x = recentre(ca.x, ctl.thx, L); ca.y = recentre(ca.y, ctl.thy, L); ca.z = recentre(ca.z, ctl.thz, L);
                cb.x = recentre(cb.x, ctl.thx, L); cb.y = recentre(cb.y, ctl.thy, L); cb.z = recentre(cb.z, ctl.thz, L);
            }
            if (SQUARE_W) { ca.w *= ca.w; cb.w *= cb.w; }
            slotp[pr] = make_float4(ca.x, cb.x, ca.y, cb.y);
            if (NEED_W) slotp[SPH_CH / 2 + pr] = make_float4(ca.z, cb.z, ca.w, cb.w);
            else slotp[SPH_CH / 2 + pr] = make_float4(ca.z, cb.z, 0.f, 0.f); // w is never read: its registers are free during the tests
            if (gidx) reinterpret_cast<uint2 *>(gidx)[pr] = make_uint2(G.j[2 * r], G.j[2 * r + 1]);
        }
    }
    __syncwarp();
}

// Lane layout of a group of g actives: lane = a + g * s with a < g the active and s < f the candidate
// stream; f is the largest divisor of SPH_CH / 2 (candidate pairs per chunk) with g * f <= 32, so that
// every chunk splits evenly over the streams.
__device__ __forceinline__ int streams_for(int g)
{
    int f = 32 / g;
    while ((SPH_CH / 2) % f) f--;
    return f;
}
