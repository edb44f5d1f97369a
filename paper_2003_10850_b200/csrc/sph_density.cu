// sph_density.cu -- steps a5-a9: neighbour gather, density sum with its h-derivative and the counts,
// safeguarded Newton iteration of the support radius (all inside ONE persistent kernel: particles do
// not couple, so a group iterates to convergence on its own), finalise and scatter.
//
// "computes particle densities by multiple iterations" (§1); the paper's GPU loop
// "performs a tree walk and neighbour interactions in chunks" of N_chunk = 32 (§2.4);
// formulas: DESIGN.md readings R1-R7.
#include "sph_gather.cuh"

#define DENS_TILE 2048 // candidates per shared-memory tile (float4 each, 32 KB)

namespace {

struct DensArgs {
    const SphNode *nodes;
    uint32_t n_nodes;
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

// w(q) and d(q) = 3 w + q w' from u = q^2 (R1); -sigma H^-4 d is dW/dH
template <int KERNEL>
__device__ __forceinline__ void kern_wd(float u, float &w, float &d)
{
    float q = u * rsqrtf(fmaxf(u, 1e-30f));
    if (KERNEL == SPH_KERNEL_CUBIC) {
        float t = 1.f - q, t2 = t * t;
        float wa = fmaf(u, fmaf(6.f, q, -6.f), 1.f), da = fmaf(u, fmaf(36.f, q, -30.f), 3.f);
        float wb = 2.f * t2 * t, db = 6.f * t2 * fmaf(-2.f, q, 1.f);
        bool in = q <= 0.5f;
        w = in ? wa : wb;
        d = in ? da : db;
    } else {
        float t = 1.f - q, t2 = t * t, t4 = t2 * t2, t7 = t4 * t2 * t;
        float p1 = fmaf(q, fmaf(q, fmaf(32.f, q, 25.f), 8.f), 1.f);
        float p2 = fmaf(q, fmaf(16.f, q, 7.f), 1.f);
        w = t7 * t * p1;
        d = t7 * fmaf(3.f * t, p1, -22.f * u * p2);
    }
}

struct DensShared {
    WalkShared ws;
    float ax[SPH_MAXB], ay[SPH_MAXB], az[SPH_MAXB], aH[SPH_MAXB];
    uint32_t aslot[SPH_MAXB];
    double aS[SPH_MAXB], aD[SPH_MAXB], aR[SPH_MAXB], aDR[SPH_MAXB];
    double lo[SPH_MAXB], hi[SPH_MAXB];
    int aCnt[SPH_MAXB], it[SPH_MAXB];
    int ulist[SPH_MAXB];
    int n_u, g;
    float q[SPH_WARPS][SPH_ABLK][SPH_QCAP];
    float qm[SPH_WARPS][SPH_ABLK][SPH_QCAP];
};

// One unit: A actives (ulist[ub..ub+A)) against tile[c0..c1). Lanes stride over the candidates, every
// lane tests its candidate against the A actives held in registers; hits are compacted into a per-
// (warp, active) ring buffer and evaluated 32 at a time so that the kernel arithmetic runs on full warps.
template <int KERNEL, bool HAS_MASS, bool PAIRWRAP, int A>
__device__ __forceinline__ void dens_unit(DensShared &sh, const float4 *__restrict__ tile, int c0, int c1, int ub, float L)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt = lanemask_lt();
    float xi[A], yi[A], zi[A], h2[A], ih2[A];
    float s0[A], s1[A], r0[A], r1[A];
    int cn[A];
    unsigned tail[A], head[A];
    int k[A];
    const float tx = sh.ws.thr[0], ty = sh.ws.thr[1], tz = sh.ws.thr[2];
#pragma unroll
    for (int a = 0; a < A; a++) {
        k[a] = sh.ulist[ub + a];
        float x = sh.ax[k[a]], y = sh.ay[k[a]], z = sh.az[k[a]], H = sh.aH[k[a]];
        xi[a] = x - ((x >= tx) ? L : 0.f);
        yi[a] = y - ((y >= ty) ? L : 0.f);
        zi[a] = z - ((z >= tz) ? L : 0.f);
        h2[a] = H * H;
        ih2[a] = 1.f / h2[a];
        s0[a] = s1[a] = r0[a] = r1[a] = 0.f;
        cn[a] = 0;
        tail[a] = head[a] = 0u;
    }
    float *qw = &sh.q[warp][0][0];
    float *qmw = &sh.qm[warp][0][0];

    auto flush = [&](int a, int nvalid) {
        __syncwarp();
        if (lane < nvalid) {
            unsigned p = (head[a] + lane) & (SPH_QCAP - 1);
            float u = qw[a * SPH_QCAP + p] * ih2[a];
            float w, d;
            kern_wd<KERNEL>(u, w, d);
            s0[a] += w;
            s1[a] += d;
            if (HAS_MASS) {
                float m = qmw[a * SPH_QCAP + p];
                r0[a] = fmaf(m, w, r0[a]);
                r1[a] = fmaf(m, d, r1[a]);
            }
        }
        __syncwarp();
    };

    for (int j0 = c0; j0 < c1; j0 += 32) {
        int j = j0 + lane;
        float4 c = (j < c1) ? tile[j] : make_float4(SPH_NANF, SPH_NANF, SPH_NANF, 0.f);
#pragma unroll
        for (int a = 0; a < A; a++) {
            float dx, dy, dz;
            if (PAIRWRAP) {
                dx = image_diff(xi[a], c.x, L); dy = image_diff(yi[a], c.y, L); dz = image_diff(zi[a], c.z, L);
            } else {
                dx = xi[a] - c.x; dy = yi[a] - c.y; dz = zi[a] - c.z;
            }
            float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            bool hit = r2 < h2[a];
            unsigned m = __ballot_sync(FULLMASK, hit);
            if (m) {
                if (hit) {
                    unsigned p = (tail[a] + __popc(m & lt)) & (SPH_QCAP - 1);
                    qw[a * SPH_QCAP + p] = r2;
                    if (HAS_MASS) qmw[a * SPH_QCAP + p] = c.w;
                }
                int nh = __popc(m);
                tail[a] += nh;
                cn[a] += nh;
                if (tail[a] - head[a] >= 32u) {
                    flush(a, 32);
                    head[a] += 32u;
                }
            }
        }
    }
#pragma unroll
    for (int a = 0; a < A; a++) {
        int rem = (int)(tail[a] - head[a]);
        if (rem > 0) flush(a, rem);
        double S = warp_sum_d((double)s0[a]), D = warp_sum_d((double)s1[a]);
        double R = 0, DR = 0;
        if (HAS_MASS) { R = warp_sum_d((double)r0[a]); DR = warp_sum_d((double)r1[a]); }
        if (lane == 0) {
            atomicAdd(&sh.aS[k[a]], S);
            atomicAdd(&sh.aD[k[a]], D);
            if (HAS_MASS) { atomicAdd(&sh.aR[k[a]], R); atomicAdd(&sh.aDR[k[a]], DR); }
            atomicAdd(&sh.aCnt[k[a]], cn[a]);
        }
    }
}

template <int KERNEL, bool HAS_MASS, bool PAIRWRAP>
__device__ __forceinline__ void dens_units(DensShared &sh, const float4 *tile, int tn, float L)
{
    const int warp = threadIdx.x >> 5;
    const int n_u = sh.n_u;
    UnitPlan pl = plan_units(n_u);
    int units = pl.nb * pl.parts;
    for (int un = warp; un < units; un += SPH_WARPS) {
        int b = un / pl.parts, part = un - b * pl.parts;
        int ub = (b * n_u) / pl.nb, ue = ((b + 1) * n_u) / pl.nb;
        int per = (((tn + pl.parts - 1) / pl.parts) + 31) & ~31;
        int c0 = min(part * per, tn), c1 = min(c0 + per, tn);
        int A = ue - ub;
        if (A <= 0 || c0 >= c1) continue;
        switch (A) {
        case 1: dens_unit<KERNEL, HAS_MASS, PAIRWRAP, 1>(sh, tile, c0, c1, ub, L); break;
        case 2: dens_unit<KERNEL, HAS_MASS, PAIRWRAP, 2>(sh, tile, c0, c1, ub, L); break;
        case 3: dens_unit<KERNEL, HAS_MASS, PAIRWRAP, 3>(sh, tile, c0, c1, ub, L); break;
        default: dens_unit<KERNEL, HAS_MASS, PAIRWRAP, 4>(sh, tile, c0, c1, ub, L); break;
        }
    }
}

template <int KERNEL, bool HAS_MASS>
__global__ void __launch_bounds__(SPH_THREADS) k_density(DensArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *tile = reinterpret_cast<float4 *>(smem_raw);
    __shared__ DensShared sh;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float L = a.L;
    const unsigned int n_groups = *a.n_groups;
    unsigned long long st_evals = 0, st_cands = 0, st_pairs = 0; // meaningful in thread 0 only
    unsigned int st_unconv = 0;

    for (;;) {
        __syncthreads();
        if (tid == 0) sh.g = (int)atomicAdd(&a.cnt->work, 1u);
        __syncthreads();
        const unsigned int g = (unsigned int)sh.g;
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
            sh.aslot[tid] = id;
            sh.ax[tid] = p.x; sh.ay[tid] = p.y; sh.az[tid] = p.z;
            sh.aH[tid] = a.h[id];
            sh.lo[tid] = 0.0;
            sh.hi[tid] = (double)__int_as_float(0x7f800000);
            sh.it[tid] = 0;
            sh.ulist[tid] = tid;
        }
        if (tid == 0) sh.n_u = na;
        __syncthreads();

        while (sh.n_u > 0) {
            const int n_u = sh.n_u;
            // bounding box and reach of the particles still iterating; zero their accumulators
            if (warp == 0) {
                float x0 = 3e38f, x1 = -3e38f, y0 = 3e38f, y1 = -3e38f, z0 = 3e38f, z1 = -3e38f, hm = 0.f;
                if (lane < n_u) {
                    int k = sh.ulist[lane];
                    x0 = x1 = sh.ax[k]; y0 = y1 = sh.ay[k]; z0 = z1 = sh.az[k];
                    hm = sh.aH[k];
                    sh.aS[k] = sh.aD[k] = sh.aR[k] = sh.aDR[k] = 0.0;
                    sh.aCnt[k] = 0;
                }
                x0 = warp_min(x0); x1 = warp_max(x1);
                y0 = warp_min(y0); y1 = warp_max(y1);
                z0 = warp_min(z0); z1 = warp_max(z1);
                hm = warp_max(hm);
                if (lane == 0) {
                    sh.ws.gc[0] = 0.5f * (x0 + x1); sh.ws.gh[0] = 0.5f * (x1 - x0) * (1.f + 1e-6f);
                    sh.ws.gc[1] = 0.5f * (y0 + y1); sh.ws.gh[1] = 0.5f * (y1 - y0) * (1.f + 1e-6f);
                    sh.ws.gc[2] = 0.5f * (z0 + z1); sh.ws.gh[2] = 0.5f * (z1 - z0) * (1.f + 1e-6f);
                    sh.ws.hg = hm;
                    sh.ws.sp = -1;
                }
                __syncwarp();
            }
            unsigned long long iter_cands = 0;
            bool more_walk;
            do {
                __syncthreads(); // everyone is done with the previous batch's lists
                if (warp == 0) walk_batch<false>(sh.ws, a.nodes, nullptr, L, DENS_TILE, a.n_nodes);
                __syncthreads();
                const uint32_t total = sh.ws.total;
                more_walk = sh.ws.sp > 0;
                iter_cands += total;
                for (uint32_t tb = 0; tb < total; tb += DENS_TILE) {
                    float4 *tiles[1] = {tile};
                    const float4 *srcs[1] = {a.xyzm};
                    stage_tile<1>(sh.ws, tiles, srcs, tb, DENS_TILE, L);
                    __syncthreads();
                    int tn = (int)min((uint32_t)DENS_TILE, total - tb);
                    if (sh.ws.pairwrap) dens_units<KERNEL, HAS_MASS, true>(sh, tile, tn, L);
                    else dens_units<KERNEL, HAS_MASS, false>(sh, tile, tn, L);
                    __syncthreads();
                }
            } while (more_walk);

            // a8: safeguarded Newton update (R7), one lane per particle, fp64 scalars
            if (warp == 0) {
                bool more = false, bad = false;
                int k = -1;
                if (lane < n_u) {
                    k = sh.ulist[lane];
                    const double H = (double)sh.aH[k];
                    const double S = sh.aS[k], D = sh.aD[k];
                    const int nint = sh.aCnt[k];
                    const double Nw = (4.0 * 3.14159265358979323846 / 3.0) * KernelConst<KERNEL>::sigma * S;
                    const double N = a.count_mode ? (double)nint : Nw;
                    const double nt = (double)a.n_target, tol = (double)a.n_tol;
                    int it = ++sh.it[k];
                    int flag = 0;
                    double lo = sh.lo[k], hi = sh.hi[k], Hn = H;
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
                            double s = (N == 0.0) ? smax : 1.0 - (N - nt) / (3.0 * N) * gs;
                            s = fmin(fmax(s, smin), smax);
                            Hn = H * s;
                            if (br && !(lo < Hn && Hn < hi)) Hn = cbrt(0.5 * (lo * lo * lo + hi * hi * hi));
                            Hn = fmin(Hn, 0.49999 * (double)L);
                            // the evaluation runs at fp32 H: a step below fp32 resolution cannot move it
                            if ((float)Hn == (float)H) flag = SPH_ST_STALLED;
                        }
                    }
                    sh.lo[k] = lo; sh.hi[k] = hi;
                    if (flag) { // a9: finalise and scatter to the caller's particle id
                        const uint32_t id = sh.aslot[k];
                        const double ih = 1.0 / H, ih3 = ih * ih * ih;
                        double rho, om;
                        if (HAS_MASS) {
                            rho = KernelConst<KERNEL>::sigma * ih3 * sh.aR[k];
                            om = 1.0 - sh.aDR[k] / (3.0 * sh.aR[k]);
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
                        sh.aH[k] = (float)Hn;
                        more = true;
                    }
                }
                // statistics (warp-uniform reductions)
                unsigned long long pr = (lane < n_u) ? (unsigned long long)sh.aCnt[k] : 0ull;
#pragma unroll
                for (int o = 16; o; o >>= 1) pr += __shfl_xor_sync(FULLMASK, pr, o);
                unsigned mb = __ballot_sync(FULLMASK, bad);
                unsigned mm = __ballot_sync(FULLMASK, more);
                if (lane == 0) {
                    st_evals += (unsigned long long)n_u;
                    st_cands += iter_cands * (unsigned long long)n_u;
                    st_pairs += pr;
                    st_unconv += __popc(mb);
                }
                // compact the list of particles that keep iterating
                __syncwarp();
                if (more) sh.ulist[__popc(mm & lanemask_lt())] = k;
                if (lane == 0) sh.n_u = __popc(mm);
            }
            __syncthreads();
        }
    }
    if (tid == 0) {
        if (st_evals) atomicAdd(&a.cnt->dens_evals, st_evals);
        if (st_cands) atomicAdd(&a.cnt->dens_cands, st_cands);
        if (st_pairs) atomicAdd(&a.cnt->dens_pairs, st_pairs);
        if (st_unconv) atomicAdd(&a.cnt->n_unconv, st_unconv);
    }
}

__global__ void k_reset_counters(SphCounters *c, int which)
{
    c->work = 0;
    if (which == 0) { c->n_unconv = 0; c->dens_evals = 0; c->dens_cands = 0; c->dens_pairs = 0; }
    else { c->force_cands = 0; c->force_pairs = 0; }
}

template <int KERNEL, bool HAS_MASS>
int launch(sph_ctx *ctx, const DensArgs &a, int grid)
{
    size_t dyn = sizeof(float4) * DENS_TILE;
    SPH_CUDA(ctx, cudaFuncSetAttribute(k_density<KERNEL, HAS_MASS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    k_density<KERNEL, HAS_MASS><<<grid, SPH_THREADS, dyn, ctx->stream>>>(a);
    SPH_CUDA(ctx, cudaGetLastError());
    return SPH_OK;
}

} // namespace

void sph_reset_counters(sph_ctx *ctx, int which)
{
    k_reset_counters<<<1, 1, 0, ctx->stream>>>(ctx->cnt, which);
    ctx->launches++;
}

int sph_density_launch(sph_ctx *ctx, bool subset, int64_t n_items, float n_target, float n_tol, float *h, float *rho,
                       float *omega, int32_t *ngb, int32_t *status)
{
    DensArgs a;
    a.nodes = ctx->nodes;
    a.n_nodes = (uint32_t)ctx->n_nodes;
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
    sph_reset_counters(ctx, 0);
    // persistent CTAs: enough to fill every SM at the occupancy the kernel reaches
    int64_t est_groups = subset ? n_items : ctx->n_groups;
    int grid = ctx->device_sms * 5;
    if (est_groups < grid) grid = (int)(est_groups > 0 ? est_groups : 1);
    int rc;
    cudaEventRecord(ctx->ev[2], ctx->stream);
    if (ctx->prm.kernel == SPH_KERNEL_CUBIC)
        rc = ctx->has_mass ? launch<SPH_KERNEL_CUBIC, true>(ctx, a, grid) : launch<SPH_KERNEL_CUBIC, false>(ctx, a, grid);
    else
        rc = ctx->has_mass ? launch<SPH_KERNEL_WC6, true>(ctx, a, grid) : launch<SPH_KERNEL_WC6, false>(ctx, a, grid);
    cudaEventRecord(ctx->ev[3], ctx->stream);
    ctx->ev_set[1] = true;
    ctx->launches++;
    return rc;
}
