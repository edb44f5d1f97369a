// sph_density.cu -- steps a5-a9: neighbour gather, density sum with its h-derivative and the counts,
// safeguarded Newton iteration of the support radius (all inside ONE persistent kernel: particles do
// not couple, so a group iterates to convergence on its own), finalise and scatter.
//
// "computes particle densities by multiple iterations" (§1); the paper's GPU loop
// "performs a tree walk and neighbour interactions in chunks" of N_chunk = 32 (§2.4);
// formulas: DESIGN.md readings R1-R7.
//
// Mapping: one CTA (4 warps) per group of g <= 32 active particles.  Thread =
// (active a, stream s): the f = 128/g streams split the candidate quads, threads of one stream read the
// same quad (shared-memory broadcast).  Warp 0 walks the octree once for the group; all warps stage the
// candidate runs it found in shared memory as component arrays X[], Y[], Z[] (in the group's periodic
// frame), where they STAY for every evaluation of the h iteration whose reach they cover.  Each thread
// tests four candidates per step in packed f32x2 against its own active and pushes r^2 of a hit onto
// its private queue; queued hits are evaluated in bulk so the kernel polynomial runs on converged
// warps.  No atomics on the pair path.
#include "sph_warp.cuh"

namespace {

struct DensArgs {
    const SphNode *nodes;
    const float4 *xyzm;
    const uint32_t *perm;
    const uint32_t *gstart;     // group starts (indices into the item list)
    const unsigned int *n_groups;
    const uint32_t *item_slot;  // NULL: item index == sorted slot (all active)
    uint32_t n_items, n_total;
    SphCounters *cnt;
    float L;
    float n_target, n_tol;
    int count_mode, max_iter;
    float mass_scalar;
    float *h, *rho, *omega;
    int32_t *ngb, *status;
};

template <int KERNEL>
struct KernelConst;
template <>
struct KernelConst<SPH_KERNEL_CUBIC> {
    static constexpr double sigma = 2.5464790894703253723; // 8/pi
};
template <>
struct KernelConst<SPH_KERNEL_WC6> {
    static constexpr double sigma = 6.7889530412636599415; // 1365/(64 pi)
};

// packed f32x2 helpers (sm_100: FADD2 / FMUL2 / FFMA2 do two lanes of fp32 per issue slot)
__device__ __forceinline__ float2 f2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ float2 f2(float a) { return make_float2(a, a); }

// w(q) and d(q) = 3 w + q w' for two hits at once, from u = q^2 (R1); -sigma H^-4 d is dW/dH.
// u = 1 gives w = d = 0 exactly (used to pad an odd tail).
template <int KERNEL>
__device__ __forceinline__ void kern_wd2(float2 u, float2 &w, float2 &d)
{
    float2 q;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(q.x) : "f"(u.x));
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(q.y) : "f"(u.y));
    const float2 t = __ffma2_rn(q, f2(-1.f), f2(1.f)), t2 = __fmul2_rn(t, t);
    if (KERNEL == SPH_KERNEL_CUBIC) {
        // q <= 1/2: w = 1 - 6u + 6uq, d = 3 - 30u + 36uq;  else: w = 2 t^3, d = 6 t^2 (1 - 2q)
        const float2 wa = __ffma2_rn(u, __ffma2_rn(f2(6.f), q, f2(-6.f)), f2(1.f));
        const float2 da = __ffma2_rn(u, __ffma2_rn(f2(36.f), q, f2(-30.f)), f2(3.f));
        const float2 wb = __fmul2_rn(__fmul2_rn(f2(2.f), t2), t);
        const float2 db = __fmul2_rn(__fmul2_rn(f2(6.f), t2), __ffma2_rn(f2(-2.f), q, f2(1.f)));
        w = f2(q.x <= 0.5f ? wa.x : wb.x, q.y <= 0.5f ? wa.y : wb.y);
        d = f2(q.x <= 0.5f ? da.x : db.x, q.y <= 0.5f ? da.y : db.y);
    } else {
        // w = t^8 (1 + 8q + 25q^2 + 32q^3);  3w + q w' = t^7 (3 + 21q + 29q^2 - 133q^3 - 448q^4)
        const float2 t4 = __fmul2_rn(t2, t2), t7 = __fmul2_rn(__fmul2_rn(t4, t2), t);
        const float2 p1 = __ffma2_rn(q, __ffma2_rn(q, __ffma2_rn(f2(32.f), q, f2(25.f)), f2(8.f)), f2(1.f));
        const float2 p2 = __ffma2_rn(q, __ffma2_rn(q, __ffma2_rn(q, __ffma2_rn(f2(-448.f), q, f2(-133.f)), f2(29.f)), f2(21.f)), f2(3.f));
        w = __fmul2_rn(__fmul2_rn(t7, t), p1);
        d = __fmul2_rn(t7, p2);
    }
}

// per-CTA shared memory
#define SPH_DSLOTS (SPH_DCAP + 16) // stored slots incl. the ragged tail and the all-NaN quad
template <bool HAS_MASS>
struct DensCta {
    // the staged candidates, component-wise, in the batch's frame; the ragged tail of the last quad and the
    // whole quad after it are NaN (every comparison with NaN is false)
    alignas(16) float X[SPH_DSLOTS];
    alignas(16) float Y[SPH_DSLOTS];
    alignas(16) float Z[SPH_DSLOTS];
    alignas(16) float M[HAS_MASS ? SPH_DSLOTS : 4];
    // hit queues: entry k of thread t at [k * SPH_THREADS + t] (r^2); reused for the cross-stream totals
    alignas(16) float q[SPH_QCAP * SPH_THREADS];
    float qm[HAS_MASS ? SPH_QCAP * SPH_THREADS : 4]; // mass of the hit
    WalkShared W;
    double lo[SPH_MAXB], hi[SPH_MAXB];       // bracket of the h iteration (R7)
    float ax[SPH_MAXB], ay[SPH_MAXB], az[SPH_MAXB], aH[SPH_MAXB];
    uint32_t aid[SPH_MAXB];
    int it[SPH_MAXB];
    int ulist[SPH_MAXB];                     // actives still iterating
    float walk_hg;                           // reach the segment list was walked with
    int listed;                              // W holds the group's complete segment list (one batch)
    int resident;                            // ... and the arrays hold all of its candidates (one chunk)
    int reuse;                               // this evaluation reuses the list
    unsigned int nstaged;                    // candidates in the arrays
    int n_u;
    unsigned int gnext;
};

#define SPH_QSTRIDE (4u * SPH_THREADS) // bytes between consecutive queue entries of a thread

// Per-thread state of one evaluation: thread = (active a, candidate stream s).
struct DensLane {
    float2 s, ds, r, dr; // packed partial sums: sum w, sum d, sum m w, sum m d
    float2 nx, ny, nz;   // minus the active's position in the batch's frame, duplicated for f32x2
    float xi, yi, zi;    // raw position (per-pair image path)
    float h2, ih2;       // H^2 (-1 for a dead thread: never hits), 1 / H^2
    uint32_t q0, qw;     // this thread's hit queue: base and write cursor (shared-memory addresses)
    uint32_t mofs;       // offset from a queue entry to its mass entry
    int cn;              // hits evaluated so far
};

__device__ __forceinline__ float lds_f32(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
    return v;
}

// Evaluate the newest min(n, queued) hits of every thread of the warp, two per step, without branches:
// a thread that runs out of entries evaluates u = 1, where w = d = 0 exactly (n is warp-uniform).
template <int KERNEL, bool HAS_MASS>
__device__ __forceinline__ void drain(DensLane &A, int n)
{
    const int m = min(n, (int)((A.qw - A.q0) / SPH_QSTRIDE));
    const uint32_t end = A.qw;
    uint32_t ra = end - (uint32_t)m * SPH_QSTRIDE;
    A.qw = ra;
    A.cn += m;
    const float2 ih22 = f2(A.ih2);
#pragma unroll 2
    for (int k = 0; k < n; k += 2, ra += 2u * SPH_QSTRIDE) {
        const bool v0 = ra < end, v1 = ra + SPH_QSTRIDE < end;
        const float r0 = v0 ? lds_f32(ra) : 0.f, r1 = v1 ? lds_f32(ra + SPH_QSTRIDE) : 0.f;
        float2 u = __fmul2_rn(f2(r0, r1), ih22);
        u.x = v0 ? u.x : 1.f;
        u.y = v1 ? u.y : 1.f;
        float2 w, d;
        kern_wd2<KERNEL>(u, w, d);
        A.s = __fadd2_rn(A.s, w);
        A.ds = __fadd2_rn(A.ds, d);
        if (HAS_MASS) {
            const float2 mj = f2(v0 ? lds_f32(ra + A.mofs) : 0.f, v1 ? lds_f32(ra + SPH_QSTRIDE + A.mofs) : 0.f);
            A.r = __ffma2_rn(mj, w, A.r);
            A.dr = __ffma2_rn(mj, d, A.dr);
        }
    }
}

// queue capacity: room for `need` more hits in every thread of the warp, else evaluate queued hits first.
// Only as many as the emptiest live queue holds (every lane busy), unless more room is needed.
template <int KERNEL, bool HAS_MASS>
__device__ __forceinline__ void make_room(DensLane &A, bool live, int need)
{
    const int cnt = (int)((A.qw - A.q0) / SPH_QSTRIDE);
    const int mx = __reduce_max_sync(FULLMASK, cnt);
    if (mx + need > SPH_QCAP) {
        const int mn = __reduce_min_sync(FULLMASK, live ? cnt : 0x7fffffff);
        drain<KERNEL, HAS_MASS>(A, max(min(mn, mx), mx + need - SPH_QCAP));
    }
}

// one candidate against this thread's active: a hit pushes r^2 (and the mass) onto the queue
template <bool HAS_MASS>
__device__ __forceinline__ void push_if(const DensLane &A, uint32_t &qw, float r2, float m)
{
    if (r2 < A.h2) {
        sts_f32(qw, r2);
        if (HAS_MASS) sts_f32(qw + A.mofs, m);
        qw += SPH_QSTRIDE;
    }
}

// Test the nq candidate quads staged in shared memory against this thread's active: thread (a, s) takes
// the quads s, s + f, s + 2f, ... (past the end: the all-NaN quad nq); the four distances of a quad come
// out of two packed f32x2 chains.
template <int KERNEL, bool HAS_MASS, bool PAIRWRAP>
__device__ __forceinline__ void consume(const DensCta<HAS_MASS> &C, DensLane &A, int nq, int s, int f, bool live, float L)
{
    const float4 *X4 = reinterpret_cast<const float4 *>(C.X), *Y4 = reinterpret_cast<const float4 *>(C.Y);
    const float4 *Z4 = reinterpret_cast<const float4 *>(C.Z), *M4 = reinterpret_cast<const float4 *>(C.M);
    const int steps = (nq + f - 1) / f; // CTA-uniform
    int qd = s, qi = min(qd, nq);
    // software pipeline: the next quad is in flight while this one is tested
    float4 nx = X4[qi], ny = Y4[qi], nz = Z4[qi], nm = HAS_MASS ? M4[qi] : make_float4(0.f, 0.f, 0.f, 0.f);
    for (int t0 = 0; t0 < steps; t0 += SPH_QSTEP) {
        const int nt = min(SPH_QSTEP, steps - t0);
        make_room<KERNEL, HAS_MASS>(A, live, 4 * nt);
        uint32_t qw = A.qw;
#pragma unroll 2
        for (int t = 0; t < nt; t++) {
            const float4 x = nx, y = ny, z = nz, m = nm;
            qd += f;
            qi = min(qd, nq);
            nx = X4[qi]; ny = Y4[qi]; nz = Z4[qi];
            if (HAS_MASS) nm = M4[qi];
            float2 ra, rb;
            if (PAIRWRAP) {
                const float dx0 = image_diff(A.xi, x.x, L), dx1 = image_diff(A.xi, x.y, L);
                const float dx2 = image_diff(A.xi, x.z, L), dx3 = image_diff(A.xi, x.w, L);
                const float dy0 = image_diff(A.yi, y.x, L), dy1 = image_diff(A.yi, y.y, L);
                const float dy2 = image_diff(A.yi, y.z, L), dy3 = image_diff(A.yi, y.w, L);
                const float dz0 = image_diff(A.zi, z.x, L), dz1 = image_diff(A.zi, z.y, L);
                const float dz2 = image_diff(A.zi, z.z, L), dz3 = image_diff(A.zi, z.w, L);
                ra = f2(fmaf(dz0, dz0, fmaf(dy0, dy0, dx0 * dx0)), fmaf(dz1, dz1, fmaf(dy1, dy1, dx1 * dx1)));
                rb = f2(fmaf(dz2, dz2, fmaf(dy2, dy2, dx2 * dx2)), fmaf(dz3, dz3, fmaf(dy3, dy3, dx3 * dx3)));
            } else {
                const float2 dxa = __fadd2_rn(f2(x.x, x.y), A.nx), dxb = __fadd2_rn(f2(x.z, x.w), A.nx);
                const float2 dya = __fadd2_rn(f2(y.x, y.y), A.ny), dyb = __fadd2_rn(f2(y.z, y.w), A.ny);
                const float2 dza = __fadd2_rn(f2(z.x, z.y), A.nz), dzb = __fadd2_rn(f2(z.z, z.w), A.nz);
                ra = __ffma2_rn(dza, dza, __ffma2_rn(dya, dya, __fmul2_rn(dxa, dxa)));
                rb = __ffma2_rn(dzb, dzb, __ffma2_rn(dyb, dyb, __fmul2_rn(dxb, dxb)));
            }
            push_if<HAS_MASS>(A, qw, ra.x, m.x);
            push_if<HAS_MASS>(A, qw, ra.y, m.y);
            push_if<HAS_MASS>(A, qw, rb.x, m.z);
            push_if<HAS_MASS>(A, qw, rb.y, m.w);
        }
        A.qw = qw;
    }
}

// Stage the candidates [lo, lo + cnt) of the walk batch's flat index space (segment k covers
// [seg_pre[k], seg_pre[k+1])) in the component arrays.  Warp w reads a quarter of the range, 32
// consecutive positions at a time (coalesced 16-byte loads): the segments that begin inside the window
// become bits of a warp-uniform mask, the segment of a position is a population count.  Candidates are
// moved into the batch's frame (recentre: exact).  The walk prunes cell by cell, so most of what it
// lists lies in the corners of cells that merely touch the group's reach: a candidate is staged only if
// it lies within the walk's reach of the group's bounding box itself (one point-to-box distance per
// candidate, instead of one distance test per candidate and ACTIVE later); the survivors are packed in
// arrival order (a ballot, a population count and one shared-memory atomic per window).
template <bool HAS_MASS>
__device__ __forceinline__ void gather_chunk(DensCta<HAS_MASS> &C, const WalkCtl &ctl, uint32_t lo, uint32_t cnt,
                                             const float4 *__restrict__ src, float L)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const WalkShared &W = C.W;
    const bool rec = !ctl.pairwrap && (ctl.thx < 1e30f || ctl.thy < 1e30f || ctl.thz < 1e30f); // CTA-uniform
    // the group's box in the batch's frame (a group lies inside one octree cell below the root, i.e. on one
    // side of L/2 on every axis; if it does not -- a root-level group of a tiny set -- nothing is filtered)
    const float hl = 0.5f * L;
    const bool strad = (W.box[0] - W.box[3] < hl && W.box[0] + W.box[3] >= hl) || (W.box[1] - W.box[4] < hl && W.box[1] + W.box[4] >= hl) ||
                       (W.box[2] - W.box[5] < hl && W.box[2] + W.box[5] >= hl);
    const bool filt = !ctl.pairwrap && !(rec && strad);
    const float bx = rec ? recentre(W.box[0], ctl.thx, L) : W.box[0], by = rec ? recentre(W.box[1], ctl.thy, L) : W.box[1];
    const float bz = rec ? recentre(W.box[2], ctl.thz, L) : W.box[2];
    const float ex = W.box[3], ey = W.box[4], ez = W.box[5];
    const float lim = filt ? W.box[6] * W.box[6] * (1.f + 1e-5f) : __int_as_float(0x7f800000);
    const uint32_t per = (((cnt + SPH_WARPS - 1) / SPH_WARPS) + 31u) & ~31u; // positions per warp, whole windows
    const uint32_t b0 = lo + min(cnt, warp * per), b1 = lo + min(cnt, (warp + 1) * per);
    int kb = seg_of(W, ctl.n_seg, b0); // warp-uniform
    for (uint32_t base = b0; base < b1; base += 32) {
        const uint32_t p = base + lane;
        const int ks = kb + 1 + lane;
        const uint32_t pre = ks < ctl.n_seg ? W.seg_pre[ks] : 0xffffffffu; // >= base: kb is the last segment that begins at or before base
        const unsigned mask = __reduce_or_sync(FULLMASK, pre < base + 32u ? 1u << (pre - base) : 0u);
        const int k = kb + __popc(mask & (0xffffffffu >> (31 - lane)));
        kb += __popc(mask);
        bool keep = false;
        float4 c = make_float4(0.f, 0.f, 0.f, 0.f);
        if (p < b1) {
            c = ldg_nc(src + (W.seg_start[k] + (p - W.seg_pre[k])));
            if (rec) { c.x = recentre(c.x, ctl.thx, L); c.y = recentre(c.y, ctl.thy, L); c.z = recentre(c.z, ctl.thz, L); }
            const float dx = fmaxf(fabsf(c.x - bx) - ex, 0.f), dy = fmaxf(fabsf(c.y - by) - ey, 0.f), dz = fmaxf(fabsf(c.z - bz) - ez, 0.f);
            keep = fmaf(dz, dz, fmaf(dy, dy, dx * dx)) <= lim;
        }
        const unsigned mk = __ballot_sync(FULLMASK, keep);
        unsigned int o = 0;
        if (lane == 0 && mk) o = atomicAdd(&C.nstaged, (unsigned int)__popc(mk));
        o = __shfl_sync(FULLMASK, o, 0) + __popc(mk & lanemask_lt());
        if (keep) {
            C.X[o] = c.x; C.Y[o] = c.y; C.Z[o] = c.z;
            if (HAS_MASS) C.M[o] = c.w;
        }
    }
}

// One evaluation of the group's g iterating actives at their current H: walk (or reuse of the resident
// set), gather, test, evaluate.  Returns the totals of the i-th iterating active in thread i (i < g).
template <int KERNEL, bool HAS_MASS>
__device__ __forceinline__ void evaluate(DensCta<HAS_MASS> &C, const DensArgs &a, int g, int evalno, double &S, double &D,
                                         double &R, double &DR, int &nint, unsigned long long &cands, unsigned long long &staged, unsigned int &walks)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float L = a.L;
    const int f = streams_for(g);
    const bool live = tid < g * f;
    const int ai = live ? tid % g : 0, s = live ? tid / g : 0;
    const float inf = __int_as_float(0x7f800000);

    DensLane A;
    {
        const int k = C.ulist[ai];
        const float H = C.aH[k];
        A.xi = C.ax[k]; A.yi = C.ay[k]; A.zi = C.az[k];
        A.h2 = live ? H * H : -1.f; // a dead thread never hits
        A.ih2 = 1.f / (H * H);
        A.s = A.ds = A.r = A.dr = f2(0.f);
        A.cn = 0;
        A.q0 = A.qw = smem_u32(C.q + tid);
        A.mofs = HAS_MASS ? smem_u32(C.qm) - smem_u32(C.q) : 0u;
    }
    // warp 0 (thread i < g holds active i): bounding box and reach of the actives still iterating; the
    // segment list of the previous evaluation stays valid if it was complete and the reach has not
    // grown -- the actives still iterating are a subset (their bounding box lies inside the old one), so
    // the old list and its frame cover this evaluation; if its candidates fitted in shared memory they
    // are still there, too.
    if (warp == 0) {
        const bool has = lane < g;
        const float hg = warp_max(has ? C.aH[C.ulist[lane]] : 0.f);
        const bool reuse = C.listed && hg <= C.walk_hg;
        if (!reuse) {
            // after the first evaluation H is within a few per cent of its final value: reach a little
            // farther than needed, so that the evaluations that follow find the list still valid
            const float hgw = evalno > 0 ? hg * (1.f + SPH_REWALK_MARGIN) : hg;
            publish_box(C.W, has, A.xi, A.yi, A.zi, hgw);
            if (lane == 0) C.walk_hg = hgw;
        }
        if (lane == 0) C.reuse = reuse ? 1 : 0;
    }
    __syncthreads();
    const bool reuse = C.reuse != 0;
    if (!reuse) { walk_cta<false>(C.W, a.nodes, nullptr, L, true); walks++; }
    bool first = true, onechunk = false;
    for (;;) {
        const WalkCtl ctl = walk_result(C.W);
        // this thread's active in the batch's frame
        A.nx = f2(-(ctl.pairwrap ? A.xi : recentre(A.xi, ctl.thx, L)));
        A.ny = f2(-(ctl.pairwrap ? A.yi : recentre(A.yi, ctl.thy, L)));
        A.nz = f2(-(ctl.pairwrap ? A.zi : recentre(A.zi, ctl.thz, L)));
        const uint32_t nch = (ctl.total + SPH_DCAP - 1) / SPH_DCAP;
        const bool keep = reuse && C.resident; // the candidates themselves are still staged
        for (uint32_t c = 0; c < nch; c++) {
            const uint32_t lo = c * SPH_DCAP, cnt = min((uint32_t)SPH_DCAP, ctl.total - lo);
            if (!keep) {
                if (tid == 0) C.nstaged = 0;
                __syncthreads();
                gather_chunk<HAS_MASS>(C, ctl, lo, cnt, a.xyzm, L);
                __syncthreads();
                const uint32_t ns = C.nstaged;
                if (tid < 8) { // the ragged tail of the last quad and the quad after it
                    C.X[ns + tid] = SPH_NANF; C.Y[ns + tid] = 0.f; C.Z[ns + tid] = 0.f;
                    if (HAS_MASS) C.M[ns + tid] = 0.f;
                }
                __syncthreads();
                staged += cnt;
            }
            const uint32_t ns = C.nstaged;
            cands += ns;
            const int nq = (int)((ns + 3u) >> 2);
            if (ctl.pairwrap) consume<KERNEL, HAS_MASS, true>(C, A, nq, s, f, live, L);
            else consume<KERNEL, HAS_MASS, false>(C, A, nq, s, f, live, L);
            if (c + 1 < nch || ctl.sp > 0) __syncthreads(); // the arrays are about to be overwritten
        }
        onechunk = first && nch == 1;
        if (reuse || ctl.sp <= 0) break;
        first = false;
        walk_cta<false>(C.W, a.nodes, nullptr, L, false);
    }
    if (!reuse && tid == 0) {
        C.listed = first ? 1 : 0;              // complete in one batch
        C.resident = first && onechunk ? 1 : 0;  // ... and in one chunk
    }

    drain<KERNEL, HAS_MASS>(A, __reduce_max_sync(FULLMASK, (int)((A.qw - A.q0) / SPH_QSTRIDE)));
    // cross-stream totals through shared memory (the queues are empty now): fp64, ascending stream order
    __syncthreads();
    double *pS = reinterpret_cast<double *>(C.q), *pD = pS + SPH_THREADS, *pR = pD + SPH_THREADS, *pDR = pR + SPH_THREADS;
    int *pn = reinterpret_cast<int *>(pDR + SPH_THREADS);
    pS[tid] = (double)A.s.x + (double)A.s.y;
    pD[tid] = (double)A.ds.x + (double)A.ds.y;
    if (HAS_MASS) { pR[tid] = (double)A.r.x + (double)A.r.y; pDR[tid] = (double)A.dr.x + (double)A.dr.y; }
    pn[tid] = A.cn;
#ifdef SPH_DIAG
    {
        const int mxh = __reduce_max_sync(FULLMASK, A.cn), smh = __reduce_add_sync(FULLMASK, A.cn);
        const int nl = __popc(__ballot_sync(FULLMASK, live));
        if (lane == 0 && nl) {
            const int b = evalno < 2 ? 0 : 1;
            atomicAdd(&a.cnt->lvl_begin[2 * b], (unsigned)mxh * nl);   // reuse dead index counters as scratch
            atomicAdd(&a.cnt->lvl_done[2 * b], (unsigned)smh);
            atomicAdd(&a.cnt->lvl_begin[2 * b + 1], (unsigned)mxh * 32);
        }
    }
#endif
    __syncthreads();
    S = D = R = DR = 0.0;
    nint = 0;
    if (tid < g) {
        for (int t = tid; t < g * f; t += g) {
            S += pS[t]; D += pD[t]; nint += pn[t];
            if (HAS_MASS) { R += pR[t]; DR += pDR[t]; }
        }
    }
    __syncthreads(); // the totals are read before the next evaluation pushes onto the queues
}

template <int KERNEL, bool HAS_MASS>
__global__ void __launch_bounds__(SPH_THREADS, SPH_CTAS) k_density(DensArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    DensCta<HAS_MASS> &C = *reinterpret_cast<DensCta<HAS_MASS> *>(smem_raw);
    if (a.cnt->bad_ids) return; // an active id was out of range: compute nothing (uniform over the grid)
    const unsigned int n_groups = *a.n_groups;
    unsigned long long st_evals = 0, st_cands = 0, st_pairs = 0, st_staged = 0; // meaningful in thread 0 only
    unsigned int st_unconv = 0, st_walks = 0, st_gevals = 0;
    for (;;) {
        __syncthreads(); // the previous group's shared state is dead
        if (tid == 0) C.gnext = atomicAdd(&a.cnt->work, 1u);
        __syncthreads();
        const unsigned int g = C.gnext;
        if (g >= n_groups) break;
        const uint32_t i0 = a.gstart[g];
        const uint32_t i1 = (g + 1 < n_groups) ? a.gstart[g + 1] : a.n_items;
        const int na = (int)(i1 - i0);
        SPH_ASSERT(i1 > i0 && i1 <= a.n_items && na <= SPH_MAXB);
        if (tid < na) {
            uint32_t slot = a.item_slot ? a.item_slot[i0 + tid] : i0 + tid;
            SPH_ASSERT(slot < a.n_total);
            float4 p = a.xyzm[slot];
            uint32_t id = a.perm[slot];
            C.aid[tid] = id;
            C.ax[tid] = p.x; C.ay[tid] = p.y; C.az[tid] = p.z;
            C.aH[tid] = a.h[id];
            C.lo[tid] = 0.0;
            C.hi[tid] = (double)__int_as_float(0x7f800000);
            C.it[tid] = 0;
            C.ulist[tid] = tid;
        }
        if (tid == 0) { C.resident = 0; C.listed = 0; }
        __syncthreads();
        int n_u = na, evalno = 0;
        while (n_u > 0) {
            double S, D, R, DR;
            int nint;
            unsigned long long cands = 0;
            evaluate<KERNEL, HAS_MASS>(C, a, n_u, evalno, S, D, R, DR, nint, cands, st_staged, st_walks);
            st_gevals++;

            if (warp == 0) {
                // a8: safeguarded Newton update (R7), one thread per particle, fp64 scalars
                bool more = false, bad = false;
                int k = -1;
                if (lane < n_u) {
                    k = C.ulist[lane];
                    const double H = (double)C.aH[k];
                    const double Nw = (4.0 * 3.14159265358979323846 / 3.0) * KernelConst<KERNEL>::sigma * S;
                    const double N = a.count_mode ? (double)nint : Nw;
                    const double nt = (double)a.n_target, tol = (double)a.n_tol;
                    int it = ++C.it[k];
                    int flag = 0;
                    double lo = C.lo[k], hi = C.hi[k], Hn = H;
                    if (fabs(N - nt) <= tol) flag = SPH_ST_CONVERGED;
                    else if (it >= a.max_iter) flag = SPH_ST_NOTCONV;
                    else {
                        if (N < nt) { if (H > lo) lo = H; } else { if (H < hi) hi = H; }
                        bool br = isfinite(hi) && lo > 0.0;
                        if (br && hi - lo <= 1e-6 * lo) flag = SPH_ST_BRACKET;
                        else {
                            // g = 1/(1 + H D'/(3 S')) with D' = -sigma H^-4 D, S' = sigma H^-3 S  ->  1/(1 - D/(3S))
                            double gs = 1.0 / (1.0 - D / (3.0 * S));
                            if (!(gs > 0.0 && gs < 4.0) || N == 0.0) gs = 1.0;
                            const double smin = 0.79370052598409973738, smax = 1.25992104989487316476;
                            // Newton step on ln N(ln H): d ln N / d ln H = 3 / gs  (R7)
                            double sc = (N == 0.0) ? smax : pow(nt / N, gs / 3.0);
                            sc = fmin(fmax(sc, smin), smax);
                            Hn = H * sc;
                            if (br && !(lo < Hn && Hn < hi)) Hn = cbrt(0.5 * (lo * lo * lo + hi * hi * hi));
                            Hn = fmin(Hn, 0.49999 * (double)a.L);
                            // the evaluation runs at fp32 H: a step below fp32 resolution cannot move it
                            if ((float)Hn == (float)H) flag = SPH_ST_STALLED;
                        }
                    }
                    C.lo[k] = lo; C.hi[k] = hi;
                    if (flag) { // a9: finalise and scatter to the caller's particle id
                        const uint32_t id = C.aid[k];
                        const double ih = 1.0 / H, ih3 = ih * ih * ih;
                        double rho, om;
                        if (HAS_MASS) {
                            rho = KernelConst<KERNEL>::sigma * ih3 * R;
                            om = 1.0 - DR / (3.0 * R);
                        } else {
                            rho = (double)a.mass_scalar * KernelConst<KERNEL>::sigma * ih3 * S;
                            om = 1.0 - D / (3.0 * S);
                        }
                        a.h[id] = (float)H;
                        a.rho[id] = (float)rho;
                        a.omega[id] = (float)om;
                        a.ngb[id] = nint;
                        if (a.status) a.status[id] = it | flag;
                        bad = flag != SPH_ST_CONVERGED;
                    } else {
                        C.aH[k] = (float)Hn;
                        more = true;
                    }
                }
                // statistics (warp-uniform reductions)
                unsigned long long pr = (lane < n_u) ? (unsigned long long)nint : 0ull;
#pragma unroll
                for (int o = 16; o; o >>= 1) pr += __shfl_xor_sync(FULLMASK, pr, o);
                const unsigned mb = __ballot_sync(FULLMASK, bad);
                const unsigned mm = __ballot_sync(FULLMASK, more);
                st_evals += (unsigned long long)n_u;
                st_cands += cands * (unsigned long long)n_u;
                st_pairs += pr;
                st_unconv += __popc(mb);
                // compact the list of particles that keep iterating
                __syncwarp();
                if (more) C.ulist[__popc(mm & lanemask_lt())] = k;
                if (lane == 0) C.n_u = __popc(mm);
            }
            __syncthreads();
            n_u = C.n_u;
            evalno++;
        }
    }
    if (tid == 0) {
        if (st_evals) atomicAdd(&a.cnt->dens_evals, st_evals);
        if (st_cands) atomicAdd(&a.cnt->dens_cands, st_cands);
        if (st_pairs) atomicAdd(&a.cnt->dens_pairs, st_pairs);
        if (st_unconv) atomicAdd(&a.cnt->n_unconv, st_unconv);
        atomicAdd(&a.cnt->dens_group_evals, (unsigned long long)st_gevals);
        atomicAdd(&a.cnt->dens_walks, (unsigned long long)st_walks);
        atomicAdd(&a.cnt->dens_staged, st_staged);
    }
}

__global__ void k_reset_counters(SphCounters *c, int which, bool subset)
{
    c->work = 0;
    if (!subset) c->bad_ids = 0; // no active list in this call
    if (which == 0) { c->n_unconv = 0; c->dens_evals = 0; c->dens_cands = 0; c->dens_pairs = 0; c->dens_group_evals = 0; c->dens_walks = 0; c->dens_staged = 0; }
    else { c->force_cands = 0; c->force_pairs = 0; c->force_staged = 0; }
}

template <int KERNEL, bool HAS_MASS>
int launch(sph_ctx *ctx, const DensArgs &a, int64_t est_groups)
{
    size_t dyn = sizeof(DensCta<HAS_MASS>);
    auto kfn = k_density<KERNEL, HAS_MASS>;
    SPH_CUDA(ctx, cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    int per_sm = 1;
    SPH_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kfn, SPH_THREADS, dyn));
    if (per_sm < 1) return sph_fail(ctx, SPH_E_INTERNAL, "k_density does not fit on an SM");
    // persistent CTAs: every SM filled to the occupancy the kernel reaches
    int64_t grid = (int64_t)ctx->device_sms * per_sm;
    if (est_groups < grid) grid = est_groups > 0 ? est_groups : 1;
    kfn<<<(int)grid, SPH_THREADS, dyn, ctx->stream>>>(a);
    SPH_CUDA(ctx, cudaGetLastError());
    return SPH_OK;
}

} // namespace

void sph_reset_counters(sph_ctx *ctx, int which, bool subset)
{
    k_reset_counters<<<1, 1, 0, ctx->stream>>>(ctx->cnt, which, subset);
    ctx->launches++;
}

int sph_density_launch(sph_ctx *ctx, bool subset, int64_t n_items, float n_target, float n_tol, float *h, float *rho,
                       float *omega, int32_t *ngb, int32_t *status)
{
    DensArgs a;
    a.nodes = ctx->nodes;
    a.xyzm = ctx->xyzm;
    a.perm = ctx->perm;
    a.gstart = subset ? ctx->agrp_start : ctx->grp_start;
    a.n_groups = subset ? &ctx->cnt->n_agroups : &ctx->cnt->n_groups;
    a.item_slot = subset ? ctx->act_slot : nullptr;
    a.n_items = (uint32_t)n_items;
    a.n_total = (uint32_t)ctx->n;
    a.cnt = ctx->cnt;
    a.L = ctx->prm.box;
    a.n_target = n_target;
    a.n_tol = n_tol;
    a.count_mode = ctx->prm.count_mode;
    a.max_iter = ctx->prm.max_iter;
    a.mass_scalar = ctx->mass_scalar;
    a.h = h; a.rho = rho; a.omega = omega; a.ngb = ngb; a.status = status;
    sph_reset_counters(ctx, 0, subset);
    int64_t est_groups = subset ? n_items : ctx->n_groups;
    int rc;
    cudaEventRecord(ctx->ev[2], ctx->stream);
    if (ctx->prm.kernel == SPH_KERNEL_CUBIC)
        rc = ctx->has_mass ? launch<SPH_KERNEL_CUBIC, true>(ctx, a, est_groups) : launch<SPH_KERNEL_CUBIC, false>(ctx, a, est_groups);
    else
        rc = ctx->has_mass ? launch<SPH_KERNEL_WC6, true>(ctx, a, est_groups) : launch<SPH_KERNEL_WC6, false>(ctx, a, est_groups);
    cudaEventRecord(ctx->ev[3], ctx->stream);
    ctx->ev_set[1] = true;
    ctx->launches++;
    return rc;
}
