// sph_warp.cuh -- device code shared by the warp-per-group gather kernels (steps a5/a6):
// per-warp octree walk that emits candidate leaf segments, and the per-warp shared-memory ring that
// the candidate segments are streamed into by 1-D bulk copies (TMA, cp.async.bulk + mbarrier).
//
// One WARP owns one group of <= 32 active particles that are consecutive in the sorted order inside
// one octree leaf -- the paper's "tree walk over groups of one or more active particles"
// (§1).  Warps never synchronise with one another: walk latency of one group hides
// behind the pair arithmetic of the others.  The ring chunk plays the role of the paper's N_chunk
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
// mbarrier / bulk-copy primitives (sm_90+; SASS: SYNCS.*, UBLKCP)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void sts_f32(uint32_t addr, float v)
{
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ void sts_u32(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}

__device__ __forceinline__ uint32_t lds_u32(uint32_t addr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr) : "memory");
    return v;
}

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// global -> shared 1-D bulk copy; bytes % 16 == 0, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void fence_proxy_async()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
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
// Candidate ring of one warp: SPH_NSLOT slots of SPH_CH candidates per streamed array.  A batch's
// candidates form one flat index space [0, total) (segment k covers [seg_pre[k], seg_pre[k+1])); chunk c
// = flat range [c*CH, c*CH+CH) lands in slot (nfill % NSLOT).  Each segment piece inside the chunk is
// one bulk copy issued by one lane; the slot's mbarrier completes when all its bytes have arrived.
template <int NARR>
struct RingCtl { // warp-uniform registers
    uint32_t nfill, ncons; // chunks filled / consumed since kernel start (slot + parity derive from them)
    int kseg;              // first segment that overlaps the next chunk to fill
};

template <int NARR>
__device__ __forceinline__ void ring_fill(const WarpWalk &ws, const WalkCtl &ctl, RingCtl<NARR> &rc, float4 *ring,
                                          uint64_t *bars, const float4 *const (&src)[NARR], uint32_t chunk,
                                          uint32_t *gidx = nullptr /* [NSLOT*CH]: sorted slot of every ring entry */)
{
    const int lane = threadIdx.x & 31;
    const uint32_t lo = chunk * SPH_CH, hi = min(lo + SPH_CH, ctl.total);
    const uint32_t slot = rc.nfill % SPH_NSLOT;
    uint64_t *bar = bars + slot;
    fence_proxy_async(); // the lanes' generic-proxy writes to the slot (slot_prepare) precede the bulk copies
    __syncwarp();        // every lane is done reading the slot's previous contents
    if (lane == 0) mbar_expect_tx(bar, (hi - lo) * 16u * NARR);
    int k0 = rc.kseg;
    for (;;) {
        int k = k0 + lane;
        bool in = k < ctl.n_seg;
        uint32_t p0 = in ? ws.seg_pre[k] : 0xffffffffu, p1 = in ? ws.seg_pre[k + 1] : 0xffffffffu;
        uint32_t a = max(p0, lo), b = min(p1, hi);
        if (in && a < b) {
            const uint32_t g = ws.seg_start[k] + (a - p0);
#pragma unroll
            for (int r = 0; r < NARR; r++)
                bulk_g2s(ring + (size_t)(r * SPH_NSLOT + slot) * SPH_CH + (a - lo), src[r] + g, (b - a) * 16u, bar);
            if (gidx)
                for (uint32_t e = 0; e < b - a; e++) gidx[slot * SPH_CH + (a - lo) + e] = g + e;
        }
        // first segment of this window that reaches beyond the chunk = first segment of the next chunk
        unsigned m = __ballot_sync(FULLMASK, in && p1 > hi);
        if (m) { k0 += __ffs(m) - 1; break; }
        k0 += 32;
        if (k0 >= ctl.n_seg) { k0 = ctl.n_seg; break; }
    }
    rc.kseg = k0;
    rc.nfill++;
}

// wait for the next chunk; returns its slot
template <int NARR>
__device__ __forceinline__ uint32_t ring_wait(RingCtl<NARR> &rc, uint64_t *bars)
{
    const uint32_t slot = rc.ncons % SPH_NSLOT, parity = (rc.ncons / SPH_NSLOT) & 1u;
    mbar_wait(bars + slot, parity);
    rc.ncons++;
    return slot;
}

// After a chunk has landed: bring the slot into the layout the test loops read.  Candidates 2p and 2p+1
// (two float4 (x,y,z,w)) become the pair records (x0,x1,y0,y1), (z0,z1,w0,w1) in the same 32 bytes, so
// that a lane loads register pairs ready for packed f32x2 arithmetic; coordinates move into the batch's
// frame (recentre); entries beyond the ragged tail become NaN (every comparison with NaN is false).
__device__ __forceinline__ void slot_prepare(float4 *slotp, uint32_t nval, const WalkCtl &ctl, float L)
{
    const int lane = threadIdx.x & 31;
    const float thx = ctl.pairwrap ? __int_as_float(0x7f800000) : ctl.thx;
    const float thy = ctl.pairwrap ? __int_as_float(0x7f800000) : ctl.thy;
    const float thz = ctl.pairwrap ? __int_as_float(0x7f800000) : ctl.thz;
#pragma unroll
    for (int p = lane; p < SPH_CH / 2; p += 32) {
        float4 c0 = slotp[2 * p], c1 = slotp[2 * p + 1];
        if (2u * p >= nval) c0 = make_float4(SPH_NANF, SPH_NANF, SPH_NANF, 0.f);
        if (2u * p + 1u >= nval) c1 = make_float4(SPH_NANF, SPH_NANF, SPH_NANF, 0.f);
        slotp[2 * p] = make_float4(recentre(c0.x, thx, L), recentre(c1.x, thx, L), recentre(c0.y, thy, L),
                                   recentre(c1.y, thy, L));
        slotp[2 * p + 1] = make_float4(recentre(c0.z, thz, L), recentre(c1.z, thz, L), c0.w, c1.w);
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
