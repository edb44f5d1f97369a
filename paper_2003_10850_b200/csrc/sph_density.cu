// sph_density.cu -- steps a5-a9: neighbour gather, density sum with its h-derivative and the counts,
// safeguarded Newton iteration of the support radius (all inside ONE persistent kernel: particles do
// not couple, so a group iterates to convergence on its own), finalise and scatter.
//
// "computes particle densities by multiple iterations" (§1); the paper's GPU loop
// "performs a tree walk and neighbour interactions in chunks" of N_chunk = 32 (§2.4);
// formulas: DESIGN.md readings R1-R7.
//
// Mapping: one warp per group of g <= 32 active particles.  Lane = (active a,
// stream s): the f ~ 32/g streams split every chunk of candidate pairs, lanes of one stream read the
// same pair record (shared-memory broadcast).  The warp gathers the candidate segments found by the
// walk, chunk by chunk, into its shared-memory slot (sph_warp.cuh); each lane tests two candidates per
// step in packed f32x2 against its own active and pushes r^2 of a hit onto its private queue; queued
// hits are evaluated in bulk so the kernel polynomial runs on converged warps.  No block-level
// barrier, no atomics on the pair path.
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

// per-warp shared memory
template <bool HAS_MASS>
struct DensWarp {
    float4 slot[SPH_CH];                     // one chunk of candidates as pair records
    WarpWalk ws;
    float q[SPH_NA * SPH_QCAP * 32];         // hit queues: entry k of lane l, active q of the lane, at [(q * QCAP + k) * 32 + l] (r^2)
    float qm[HAS_MASS ? SPH_NA * SPH_QCAP * 32 : 32]; // mass of the hit
    double lo[SPH_MAXB], hi[SPH_MAXB];       // bracket of the h iteration (R7)
    float ax[SPH_MAXB], ay[SPH_MAXB], az[SPH_MAXB], aH[SPH_MAXB];
    uint32_t aid[SPH_MAXB];
    int it[SPH_MAXB];
    int ulist[SPH_MAXB];                     // actives still iterating
};

// Per-lane state of one evaluation.  A lane is (active slot ap, candidate stream s) and holds SPH_NA
// actives (2 ap, 2 ap + 1): every pair record loaded from shared memory is tested against all of them,
// which halves the shared-memory reads and the loop overhead per test.
struct DensAct {         // one active of the lane
    float2 s, ds, r, dr; // packed partial sums: sum w, sum d, sum m w, sum m d
    float2 nx, ny, nz;   // minus the active's position in the batch's frame, duplicated for f32x2
    float xi, yi, zi;    // raw position (per-pair image path)
    float h2, ih2;       // H^2 (-1 for a missing active: never hits), 1 / H^2
    uint32_t q0, qw;     // this active's hit queue in this lane: base and write cursor (shared-memory addresses, stride 128 B)
    int cn;              // hits evaluated so far
};
struct DensLane {
    DensAct act[SPH_NA];
    uint32_t mofs;       // offset from a queue entry to its mass entry
    const float4 *cp;    // this stream's first pair record of the chunk
    int cstride;         // float4 elements between consecutive pair records of this stream (f)
    int steps;           // pair records per chunk for this stream (SPH_CH / 2 / f)
};

__device__ __forceinline__ float lds_f32(uint32_t addr)
{
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr) : "memory");
    return v;
}

// Evaluate the newest min(n, queued) hits of one active of every lane, two per step, without branches:
// a lane that runs out of entries evaluates u = 1, where w = d = 0 exactly (n is warp-uniform).
template <int KERNEL, bool HAS_MASS>
__device__ __forceinline__ void drain(DensAct &A, uint32_t mofs, int n)
{
    const int m = min(n, (int)((A.qw - A.q0) >> 7));
    const uint32_t end = A.qw;
    uint32_t ra = end - (uint32_t)m * 128u;
    A.qw = ra;
    A.cn += m;
    const float2 ih22 = f2(A.ih2);
#pragma unroll 2
    for (int k = 0; k < n; k += 2, ra += 256u) {
        const bool v0 = ra < end, v1 = ra + 128u < end;
        const float r0 = v0 ? lds_f32(ra) : 0.f, r1 = v1 ? lds_f32(ra + 128u) : 0.f;
        float2 u = __fmul2_rn(f2(r0, r1), ih22);
        u.x = v0 ? u.x : 1.f;
        u.y = v1 ? u.y : 1.f;
        float2 w, d;
        kern_wd2<KERNEL>(u, w, d);
        A.s = __fadd2_rn(A.s, w);
        A.ds = __fadd2_rn(A.ds, d);
        if (HAS_MASS) {
            const float2 mj = f2(v0 ? lds_f32(ra + mofs) : 0.f, v1 ? lds_f32(ra + 128u + mofs) : 0.f);
            A.r = __ffma2_rn(mj, w, A.r);
            A.dr = __ffma2_rn(mj, d, A.dr);
        }
    }
}

// queue capacity: room for `need` more hits of this active in every lane, else evaluate queued hits first
template <int KERNEL, bool HAS_MASS>
__device__ __forceinline__ void make_room(DensAct &A, uint32_t mofs, bool live, int need)
{
    const int cnt = (int)((A.qw - A.q0) >> 7);
    const int mx = __reduce_max_sync(FULLMASK, cnt);
    if (mx + need > SPH_QCAP) {
        const int mn = __reduce_min_sync(FULLMASK, live ? cnt : 0x7fffffff);
        drain<KERNEL, HAS_MASS>(A, mofs, max(mn, mx + need - SPH_QCAP));
    }
}

// Test the candidates of the gathered chunk against this lane's actives: lane (ap, s) takes the pair
// records s, s + f, s + 2f, ...; both distances of a pair come out of one packed f32x2 chain; a hit
// pushes r^2 (and the mass) onto the queue of the active it belongs to.
template <int KERNEL, bool HAS_MASS, bool PAIRWRAP>
__device__ __forceinline__ void consume_chunk(DensLane &A, bool live, float L)
{
    const float4 *cp = A.cp;
    float4 n0 = cp[0], n1 = cp[SPH_CH / 2];
    cp += A.cstride;
    for (int t0 = 0; t0 < A.steps; t0 += SPH_QSTEP) {
        const int nt = min(SPH_QSTEP, A.steps - t0);
#pragma unroll
        for (int a = 0; a < SPH_NA; a++) make_room<KERNEL, HAS_MASS>(A.act[a], A.mofs, live, 2 * nt);
        uint32_t qw[SPH_NA];
#pragma unroll
        for (int a = 0; a < SPH_NA; a++) qw[a] = A.act[a].qw;
#pragma unroll 3
        for (int t = 0; t < nt; t++) {
            const float4 c0 = n0, cz = n1; // (x0,x1,y0,y1) (z0,z1,w0,w1)
            const float2 c1 = f2(cz.x, cz.y), cm = f2(cz.z, cz.w);
            // software pipeline: the next pair record is in flight while this one is tested (past the
            // chunk's last record this reads on inside the warp's own shared memory; the value is unused)
            n0 = cp[0]; n1 = cp[SPH_CH / 2];
            cp += A.cstride;
#pragma unroll
            for (int a = 0; a < SPH_NA; a++) {
                const DensAct &P = A.act[a];
                float2 r2;
                if (PAIRWRAP) {
                    const float dx0 = image_diff(P.xi, c0.x, L), dx1 = image_diff(P.xi, c0.y, L);
                    const float dy0 = image_diff(P.yi, c0.z, L), dy1 = image_diff(P.yi, c0.w, L);
                    const float dz0 = image_diff(P.zi, c1.x, L), dz1 = image_diff(P.zi, c1.y, L);
                    r2 = f2(fmaf(dz0, dz0, fmaf(dy0, dy0, dx0 * dx0)), fmaf(dz1, dz1, fmaf(dy1, dy1, dx1 * dx1)));
                } else {
                    const float2 dx = __fadd2_rn(f2(c0.x, c0.y), P.nx), dy = __fadd2_rn(f2(c0.z, c0.w), P.ny);
                    const float2 dz = __fadd2_rn(c1, P.nz);
                    r2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
                }
                if (r2.x < P.h2) {
                    sts_f32(qw[a], r2.x);
                    if (HAS_MASS) sts_f32(qw[a] + A.mofs, cm.x);
                    qw[a] += 128u;
                }
                if (r2.y < P.h2) {
                    sts_f32(qw[a], r2.y);
                    if (HAS_MASS) sts_f32(qw[a] + A.mofs, cm.y);
                    qw[a] += 128u;
                }
            }
        }
#pragma unroll
        for (int a = 0; a < SPH_NA; a++) A.act[a].qw = qw[a];
    }
}

// what evaluate() keeps from one evaluation of a group to the next (warp-uniform registers)
struct WalkCache {
    WalkCtl ctl;
    float hg;    // reach the list was walked with
    bool valid;  // the list in shared memory is complete and reusable
    bool multi;  // scratch: a batch of the current walk has already been seen
};

// One evaluation of the group's g iterating actives at their current H: walk, gather, test, evaluate.
// Returns the totals of the i-th iterating active in lane i (i < g).
template <int KERNEL, bool HAS_MASS>
__device__ __forceinline__ void evaluate(DensWarp<HAS_MASS> &W, const DensArgs &a, int g, WalkCache &wc, double &S,
                                         double &D, double &R, double &DR, int &nint, unsigned long long &cands)
{
    const int lane = threadIdx.x & 31;
    const float L = a.L;
    const int gp = (g + SPH_NA - 1) / SPH_NA; // active slots: lane = ap + gp * s
    const int f = streams_for(gp);
    const bool live = lane < gp * f;
    const int ap = live ? lane % gp : 0, s = live ? lane / gp : 0;
    const float inf = __int_as_float(0x7f800000);

    DensLane A;
    A.mofs = HAS_MASS ? smem_u32(W.qm) - smem_u32(W.q) : 0u;
    A.cp = W.slot + s;
    A.cstride = f;
    A.steps = (SPH_CH / 2) / f;
    // bounding box and reach of the actives still iterating
    float x0 = inf, x1 = -inf, y0 = inf, y1 = -inf, z0 = inf, z1 = -inf, hg = 0.f;
#pragma unroll
    for (int q = 0; q < SPH_NA; q++) {
        DensAct &P = A.act[q];
        const int i = ap * SPH_NA + q;
        const bool has = live && i < g;
        const int k = W.ulist[has ? i : 0];
        const float H = W.aH[k];
        P.xi = W.ax[k]; P.yi = W.ay[k]; P.zi = W.az[k];
        P.h2 = has ? H * H : -1.f; // a missing active never hits
        P.ih2 = 1.f / (H * H);
        P.s = P.ds = P.r = P.dr = f2(0.f);
        P.cn = 0;
        P.q0 = P.qw = smem_u32(W.q + q * SPH_QCAP * 32 + lane);
        if (has) {
            x0 = fminf(x0, P.xi); x1 = fmaxf(x1, P.xi);
            y0 = fminf(y0, P.yi); y1 = fmaxf(y1, P.yi);
            z0 = fminf(z0, P.zi); z1 = fmaxf(z1, P.zi);
            hg = fmaxf(hg, H);
        }
    }
    x0 = warp_min(x0); x1 = warp_max(x1);
    y0 = warp_min(y0); y1 = warp_max(y1);
    z0 = warp_min(z0); z1 = warp_max(z1);
    hg = warp_max(hg);
    const float gcx = 0.5f * (x0 + x1), ghx = 0.5f * (x1 - x0) * (1.f + 1e-6f);
    const float gcy = 0.5f * (y0 + y1), ghy = 0.5f * (y1 - y0) * (1.f + 1e-6f);
    const float gcz = 0.5f * (z0 + z1), ghz = 0.5f * (z1 - z0) * (1.f + 1e-6f);

    // The segment list of the group's previous evaluation is still in shared memory.  It stays valid if
    // it was complete (one batch) and the reach has not grown: the actives still iterating are a subset
    // (their bounding box lies inside the old one), so the old list and its frame cover this evaluation.
    const bool reuse = wc.valid && hg <= wc.hg;
    WalkCtl ctl = wc.ctl;
    if (!reuse) ctl.sp = -1;
    do {
        if (!reuse) walk_batch<false>(W.ws, ctl, a.nodes, nullptr, L, gcx, gcy, gcz, ghx, ghy, ghz, hg);
        cands += ctl.total;
        // this lane's actives in the batch's frame
#pragma unroll
        for (int q = 0; q < SPH_NA; q++) {
            DensAct &P = A.act[q];
            P.nx = f2(-(ctl.pairwrap ? P.xi : recentre(P.xi, ctl.thx, L)));
            P.ny = f2(-(ctl.pairwrap ? P.yi : recentre(P.yi, ctl.thy, L)));
            P.nz = f2(-(ctl.pairwrap ? P.zi : recentre(P.zi, ctl.thz, L)));
        }
        const uint32_t nch = (ctl.total + SPH_CH - 1) / SPH_CH;
        GatherCtl gc;
        gc.kseg = 0;
        // software pipeline: the loads of chunk c + 1 are in flight (in registers) while chunk c is tested
        GatherRegs G;
        if (nch) gather_load(W.ws, ctl, gc, 0, G, a.xyzm);
        for (uint32_t c = 0; c < nch; c++) {
            gather_store<false, true>(ctl, G, W.slot, nullptr, L); // (writing w even when unread measured faster: 74.6 vs 78.6 ms)
            if (c + 1 < nch) gather_load(W.ws, ctl, gc, c + 1, G, a.xyzm);
            if (ctl.pairwrap) consume_chunk<KERNEL, HAS_MASS, true>(A, live, L);
            else consume_chunk<KERNEL, HAS_MASS, false>(A, live, L);
        }
        if (!reuse) {
            wc.valid = !wc.multi && ctl.sp <= 0; // complete in its first batch
            wc.multi = true;
            wc.hg = hg;
            wc.ctl = ctl;
        }
    } while (ctl.sp > 0);

    S = D = R = DR = 0.0;
    nint = 0;
#pragma unroll
    for (int q = 0; q < SPH_NA; q++) {
        DensAct &P = A.act[q];
        drain<KERNEL, HAS_MASS>(P, A.mofs, __reduce_max_sync(FULLMASK, (int)((P.qw - P.q0) >> 7)));
        // cross-stream totals: lane ap + gp*s adds lane ap + gp*(s+d) for d = 1, 2, 4, ...
        double tS = (double)P.s.x + (double)P.s.y, tD = (double)P.ds.x + (double)P.ds.y;
        double tR = (double)P.r.x + (double)P.r.y, tDR = (double)P.dr.x + (double)P.dr.y;
        int tn = P.cn;
        for (int d = 1; d < f; d <<= 1) {
            const bool take = live && s + d < f;
            const int from = take ? lane + gp * d : lane;
            const double uS = __shfl_sync(FULLMASK, tS, from), uD = __shfl_sync(FULLMASK, tD, from);
            const int un = __shfl_sync(FULLMASK, tn, from);
            if (take) { tS += uS; tD += uD; tn += un; }
            if (HAS_MASS) {
                const double uR = __shfl_sync(FULLMASK, tR, from), uDR = __shfl_sync(FULLMASK, tDR, from);
                if (take) { tR += uR; tDR += uDR; }
            }
        }
        // active i = ap * SPH_NA + q sits in lane ap (stream 0): hand it to lane i
        const int src = lane / SPH_NA;
        const double oS = __shfl_sync(FULLMASK, tS, src), oD = __shfl_sync(FULLMASK, tD, src);
        const int on = __shfl_sync(FULLMASK, tn, src);
        const bool mine = lane % SPH_NA == q;
        if (mine) { S = oS; D = oD; nint = on; }
        if (HAS_MASS) {
            const double oR = __shfl_sync(FULLMASK, tR, src), oDR = __shfl_sync(FULLMASK, tDR, src);
            if (mine) { R = oR; DR = oDR; }
        }
    }
}

template <int KERNEL, bool HAS_MASS>
__global__ void __launch_bounds__(SPH_THREADS, SPH_CTAS) k_density(DensArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    DensWarp<HAS_MASS> &W = reinterpret_cast<DensWarp<HAS_MASS> *>(smem_raw)[warp];
    if (a.cnt->err | a.cnt->idx_err) return; // a precondition failed (ids, h, positions): compute nothing (uniform over the grid)
    const unsigned int n_groups = *a.n_groups;
    unsigned long long st_evals = 0, st_cands = 0, st_pairs = 0; // meaningful in lane 0 only
    unsigned int st_unconv = 0;
    unsigned int gnext = 0, gend = 0; // this warp's block of consecutive groups (neighbouring groups share candidates in L1/L2)
    for (;;) {
        if (gnext == gend) {
            if (lane == 0) gnext = atomicAdd(&a.cnt->work, (unsigned int)SPH_GBLOCK);
            gnext = __shfl_sync(FULLMASK, gnext, 0);
            if (gnext >= n_groups) break;
            gend = min(gnext + SPH_GBLOCK, n_groups);
        }
        const unsigned int g = gnext++;
        const uint32_t i0 = a.gstart[g];
        const uint32_t i1 = (g + 1 < n_groups) ? a.gstart[g + 1] : a.n_items;
        const int na = (int)(i1 - i0);
        SPH_ASSERT(i1 > i0 && i1 <= a.n_items && na <= SPH_MAXB);
        __syncwarp();
        if (lane < na) {
            uint32_t slot = a.item_slot ? a.item_slot[i0 + lane] : i0 + lane;
            SPH_ASSERT(slot < a.n_total);
            float4 p = a.xyzm[slot];
            uint32_t id = a.perm[slot];
            W.aid[lane] = id;
            W.ax[lane] = p.x; W.ay[lane] = p.y; W.az[lane] = p.z;
            W.aH[lane] = a.h[id];
            W.lo[lane] = 0.0;
            W.hi[lane] = (double)__int_as_float(0x7f800000);
            W.it[lane] = 0;
            W.ulist[lane] = lane;
        }
        __syncwarp();
        int n_u = na;
        WalkCache wc;
        wc.valid = false;
        while (n_u > 0) {
            wc.multi = false;
            double S, D, R, DR;
            int nint;
            unsigned long long cands = 0;
            evaluate<KERNEL, HAS_MASS>(W, a, n_u, wc, S, D, R, DR, nint, cands);

            // a8: safeguarded Newton update (R7), one lane per particle, fp64 scalars
            bool more = false, bad = false;
            int k = -1;
            if (lane < n_u) {
                k = W.ulist[lane];
                const double H = (double)W.aH[k];
                const double Nw = (4.0 * 3.14159265358979323846 / 3.0) * KernelConst<KERNEL>::sigma * S;
                const double N = a.count_mode ? (double)nint : Nw;
                const double nt = (double)a.n_target, tol = (double)a.n_tol;
                int it = ++W.it[k];
                int flag = 0;
                double lo = W.lo[k], hi = W.hi[k], Hn = H;
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
                W.lo[k] = lo; W.hi[k] = hi;
                if (flag) { // a9: finalise and scatter to the caller's particle id
                    const uint32_t id = W.aid[k];
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
                    W.aH[k] = (float)Hn;
                    more = true;
                }
            }
            // statistics (warp-uniform reductions)
            unsigned long long pr = (lane < n_u) ? (unsigned long long)nint : 0ull;
#pragma unroll
            for (int o = 16; o; o >>= 1) pr += __shfl_xor_sync(FULLMASK, pr, o);
            unsigned mb = __ballot_sync(FULLMASK, bad);
            unsigned mm = __ballot_sync(FULLMASK, more);
            st_evals += (unsigned long long)n_u;
            st_cands += cands * (unsigned long long)n_u;
            st_pairs += pr;
            st_unconv += __popc(mb);
            // compact the list of particles that keep iterating
            __syncwarp();
            if (more) W.ulist[__popc(mm & lanemask_lt())] = k;
            n_u = __popc(mm);
            __syncwarp();
        }
    }
    if (lane == 0) {
        if (st_evals) atomicAdd(&a.cnt->dens_evals, st_evals);
        if (st_cands) atomicAdd(&a.cnt->dens_cands, st_cands);
        if (st_pairs) atomicAdd(&a.cnt->dens_pairs, st_pairs);
        if (st_unconv) atomicAdd(&a.cnt->n_unconv, st_unconv);
    }
}

// precondition 0 < H < box / 2 on the guesses of the active particles (not finite counts as <= 0)
__global__ void k_check_h(int64_t n_items, int64_t n, const int32_t *__restrict__ active, const float *__restrict__ h, float half_box,
                          SphCounters *cnt)
{
    int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_items) return;
    int64_t id = active ? (int64_t)active[k] : k;
    if (id < 0 || id >= n) return; // (reported by the active-list pass)
    const float H = h[id];
    if (!(H > 0.f) || !(H < __int_as_float(0x7f800000))) atomicOr(&cnt->err, SPH_ERR_H);
    else if (!(H < half_box)) atomicOr(&cnt->err, SPH_ERR_HRANGE);
}

__global__ void k_reset_counters(SphCounters *c, int which, bool subset)
{
    c->work = 0;
    if (which == 0) { c->n_unconv = 0; c->dens_evals = 0; c->dens_cands = 0; c->dens_pairs = 0; }
    else { c->force_cands = 0; c->force_pairs = 0; }
}

template <int KERNEL, bool HAS_MASS>
int launch(sph_ctx *ctx, const DensArgs &a, int64_t est_groups)
{
    size_t dyn = sizeof(DensWarp<HAS_MASS>) * SPH_WARPS;
    auto kfn = k_density<KERNEL, HAS_MASS>;
    SPH_CUDA(ctx, cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    int per_sm = 1;
    SPH_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kfn, SPH_THREADS, dyn));
    if (per_sm < 1) return sph_fail(ctx, SPH_E_INTERNAL, "k_density does not fit on an SM");
    // persistent warps: every SM filled to the occupancy the kernel reaches
    int64_t grid = (int64_t)ctx->device_sms * per_sm;
    int64_t need = (est_groups + SPH_WARPS * SPH_GBLOCK - 1) / (SPH_WARPS * SPH_GBLOCK);
    if (need < grid) grid = need > 0 ? need : 1;
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

int sph_density_launch(sph_ctx *ctx, const int32_t *active, int64_t n_items, float n_target, float n_tol, float *h, float *rho,
                       float *omega, int32_t *ngb, int32_t *status)
{
    const bool subset = active != nullptr;
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
    k_check_h<<<(int)((n_items + 255) / 256), 256, 0, ctx->stream>>>(n_items, ctx->n, active, h, 0.5f * ctx->prm.box, ctx->cnt);
    ctx->launches++;
    int64_t est_groups = n_items; // (an upper bound: the group count stays on the device)
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
