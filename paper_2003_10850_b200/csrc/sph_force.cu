// sph_force.cu -- steps a5, a6, a10, a11: symmetric hydro-force pair sum (pressure gradient +
// signal-velocity artificial viscosity) and the maximum signal velocity, for the active particles.
//
// "the second one computes hydrodynamic forces" (§1); same search pattern as the density
// module (§1).  Formulas: DESIGN.md readings R8-R12.  The neighbour set is symmetric,
// r_ij < max(H_i, H_j) (R10): the walk prunes a node only if it is farther from the group than both
// the group's reach and the largest support radius inside the node.
#include "sph_gather.cuh"

#define FORCE_TILE 1024 // candidates per shared-memory tile (3 float4 each, 48 KB)

namespace {

struct ForceArgs {
    const SphNode *nodes;
    uint32_t n_nodes;
    const float *node_hmax;
    const float4 *xyzh, *vc, *raf; // sorted: (x,y,z,H) (vx,vy,vz,c) (rho, A, m, slot)
    const uint32_t *perm;
    const uint32_t *gstart;
    const unsigned int *n_groups;
    const uint32_t *item_slot;
    uint32_t n_items;
    SphCounters *cnt;
    float L, alpha;
    float *acc, *dudt, *vsig;
};

template <int KERNEL>
__device__ __forceinline__ float kern_dw(float q) // w'(q), 0 for q >= 1 (R1)
{
    float t = fmaxf(1.f - q, 0.f);
    if (KERNEL == SPH_KERNEL_CUBIC) {
        float a = q * fmaf(18.f, q, -12.f), b = -6.f * t * t;
        return q <= 0.5f ? a : b;
    } else {
        float t2 = t * t, t4 = t2 * t2, t7 = t4 * t2 * t;
        return -22.f * q * t7 * fmaf(q, fmaf(16.f, q, 7.f), 1.f);
    }
}
template <int KERNEL>
__device__ __forceinline__ float kern_sigma()
{
    return KERNEL == SPH_KERNEL_CUBIC ? 2.54647908947032537f : 6.78895304126365994f;
}

struct ForceShared {
    WalkShared ws;
    float ax[SPH_MAXB], ay[SPH_MAXB], az[SPH_MAXB], aH[SPH_MAXB];
    float aHinv[SPH_MAXB], aF4[SPH_MAXB]; // 1/H_i, sigma/H_i^4
    float avx[SPH_MAXB], avy[SPH_MAXB], avz[SPH_MAXB], ac[SPH_MAXB], arho[SPH_MAXB], aA[SPH_MAXB];
    uint32_t aslot[SPH_MAXB], aid[SPH_MAXB];
    double fx[SPH_MAXB], fy[SPH_MAXB], fz[SPH_MAXB], fdu[SPH_MAXB];
    int fvs[SPH_MAXB]; // max signal velocity as float bits (>= 0: integer order == float order)
    int aCnt[SPH_MAXB];
    int n_u, g;
    unsigned short q[SPH_WARPS][SPH_ABLK][SPH_QCAP];
};

template <int KERNEL, bool PAIRWRAP, int A>
__device__ __forceinline__ void force_unit(ForceShared &sh, const float4 *__restrict__ t0, const float4 *__restrict__ t1,
                                           const float4 *__restrict__ t2, int c0, int c1, int ub, float L, float alpha)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const unsigned lt = lanemask_lt();
    float xi[A], yi[A], zi[A], h2[A];
    float px[A], py[A], pz[A], pdu[A], pvs[A];
    int cn[A];
    unsigned tail[A], head[A];
    const float tx = sh.ws.thr[0], ty = sh.ws.thr[1], tz = sh.ws.thr[2];
#pragma unroll
    for (int a = 0; a < A; a++) {
        int k = ub + a;
        float x = sh.ax[k], y = sh.ay[k], z = sh.az[k], H = sh.aH[k];
        xi[a] = x - ((x >= tx) ? L : 0.f);
        yi[a] = y - ((y >= ty) ? L : 0.f);
        zi[a] = z - ((z >= tz) ? L : 0.f);
        h2[a] = H * H;
        px[a] = py[a] = pz[a] = pdu[a] = pvs[a] = 0.f;
        cn[a] = 0;
        tail[a] = head[a] = 0u;
    }
    unsigned short *qw = &sh.q[warp][0][0];

    auto flush = [&](int a, int nvalid) {
        __syncwarp();
        if (lane < nvalid) {
            const int k = ub + a;
            unsigned p = (head[a] + lane) & (SPH_QCAP - 1);
            int j = qw[a * SPH_QCAP + p];
            float4 P0 = t0[j], P1 = t1[j], P2 = t2[j];
            if (__float_as_uint(P2.w) != sh.aslot[k]) { // j != i
                float dx, dy, dz;
                if (PAIRWRAP) {
                    dx = image_diff(xi[a], P0.x, L); dy = image_diff(yi[a], P0.y, L); dz = image_diff(zi[a], P0.z, L);
                } else {
                    dx = xi[a] - P0.x; dy = yi[a] - P0.y; dz = zi[a] - P0.z;
                }
                float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                float rinv = rsqrtf(fmaxf(r2, 1e-37f));
                float r = r2 * rinv;
                float hinv_j = __fdividef(1.f, P0.w);
                float hj2 = hinv_j * hinv_j;
                float Fi = sh.aF4[k] * kern_dw<KERNEL>(r * sh.aHinv[k]);
                float Fj = kern_sigma<KERNEL>() * hj2 * hj2 * kern_dw<KERNEL>(r * hinv_j);
                float dvx = sh.avx[k] - P1.x, dvy = sh.avy[k] - P1.y, dvz = sh.avz[k] - P1.z;
                float vr = fmaf(dvz, dz, fmaf(dvy, dy, dvx * dx)) * rinv;
                float mu = fminf(vr, 0.f);
                float vs = sh.ac[k] + P1.w - 3.f * mu;
                float Pi = -alpha * vs * mu * __fdividef(1.f, sh.arho[k] + P2.x);
                float Fbar = 0.5f * (Fi + Fj);
                float AiFi = sh.aA[k] * Fi;
                float pv = Pi * Fbar;
                float t = P2.z * (AiFi + fmaf(P2.y, Fj, pv));
                float tr = t * rinv;
                px[a] = fmaf(-tr, dx, px[a]);
                py[a] = fmaf(-tr, dy, py[a]);
                pz[a] = fmaf(-tr, dz, pz[a]);
                pdu[a] = fmaf(P2.z * fmaf(0.5f, pv, AiFi), vr, pdu[a]);
                pvs[a] = fmaxf(pvs[a], vs);
            }
        }
        __syncwarp();
    };

    for (int j0 = c0; j0 < c1; j0 += 32) {
        int j = j0 + lane;
        float4 c = (j < c1) ? t0[j] : make_float4(SPH_NANF, SPH_NANF, SPH_NANF, 0.f);
        float hj2 = c.w * c.w;
#pragma unroll
        for (int a = 0; a < A; a++) {
            float dx, dy, dz;
            if (PAIRWRAP) {
                dx = image_diff(xi[a], c.x, L); dy = image_diff(yi[a], c.y, L); dz = image_diff(zi[a], c.z, L);
            } else {
                dx = xi[a] - c.x; dy = yi[a] - c.y; dz = zi[a] - c.z;
            }
            float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            bool hit = r2 < fmaxf(h2[a], hj2);
            unsigned m = __ballot_sync(FULLMASK, hit);
            if (m) {
                if (hit) {
                    unsigned p = (tail[a] + __popc(m & lt)) & (SPH_QCAP - 1);
                    qw[a * SPH_QCAP + p] = (unsigned short)j;
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
        double X = warp_sum_d((double)px[a]), Y = warp_sum_d((double)py[a]), Z = warp_sum_d((double)pz[a]);
        double U = warp_sum_d((double)pdu[a]);
        float V = warp_max(pvs[a]);
        if (lane == 0) {
            int k = ub + a;
            atomicAdd(&sh.fx[k], X);
            atomicAdd(&sh.fy[k], Y);
            atomicAdd(&sh.fz[k], Z);
            atomicAdd(&sh.fdu[k], U);
            atomicMax(&sh.fvs[k], __float_as_int(V));
            atomicAdd(&sh.aCnt[k], cn[a]);
        }
    }
}

template <int KERNEL, bool PAIRWRAP>
__device__ __forceinline__ void force_units(ForceShared &sh, const float4 *t0, const float4 *t1, const float4 *t2, int tn,
                                            float L, float alpha)
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
        case 1: force_unit<KERNEL, PAIRWRAP, 1>(sh, t0, t1, t2, c0, c1, ub, L, alpha); break;
        case 2: force_unit<KERNEL, PAIRWRAP, 2>(sh, t0, t1, t2, c0, c1, ub, L, alpha); break;
        case 3: force_unit<KERNEL, PAIRWRAP, 3>(sh, t0, t1, t2, c0, c1, ub, L, alpha); break;
        default: force_unit<KERNEL, PAIRWRAP, 4>(sh, t0, t1, t2, c0, c1, ub, L, alpha); break;
        }
    }
}

template <int KERNEL>
__global__ void __launch_bounds__(SPH_THREADS) k_force(ForceArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float4 *t0 = reinterpret_cast<float4 *>(smem_raw);
    float4 *t1 = t0 + FORCE_TILE;
    float4 *t2 = t1 + FORCE_TILE;
    __shared__ ForceShared sh;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const float L = a.L;
    const unsigned int n_groups = *a.n_groups;
    unsigned long long st_cands = 0, st_pairs = 0;

    for (;;) {
        __syncthreads();
        if (tid == 0) sh.g = (int)atomicAdd(&a.cnt->work, 1u);
        __syncthreads();
        const unsigned int g = (unsigned int)sh.g;
        if (g >= n_groups) break;
        const uint32_t i0 = a.gstart[g];
        const uint32_t i1 = (g + 1 < n_groups) ? a.gstart[g + 1] : a.n_items;
        const int na = (int)(i1 - i0);
        if (tid < na) {
            uint32_t slot = a.item_slot ? a.item_slot[i0 + tid] : i0 + tid;
            float4 p0 = a.xyzh[slot], p1 = a.vc[slot], p2 = a.raf[slot];
            sh.aslot[tid] = slot;
            sh.aid[tid] = a.perm[slot];
            sh.ax[tid] = p0.x; sh.ay[tid] = p0.y; sh.az[tid] = p0.z; sh.aH[tid] = p0.w;
            float hinv = 1.f / p0.w, h2i = hinv * hinv;
            sh.aHinv[tid] = hinv;
            sh.aF4[tid] = kern_sigma<KERNEL>() * h2i * h2i;
            sh.avx[tid] = p1.x; sh.avy[tid] = p1.y; sh.avz[tid] = p1.z; sh.ac[tid] = p1.w;
            sh.arho[tid] = p2.x; sh.aA[tid] = p2.y;
            sh.fx[tid] = sh.fy[tid] = sh.fz[tid] = sh.fdu[tid] = 0.0;
            sh.fvs[tid] = 0;
            sh.aCnt[tid] = 0;
        }
        if (tid == 0) sh.n_u = na;
        __syncthreads();
        if (warp == 0) {
            float x0 = 3e38f, x1 = -3e38f, y0 = 3e38f, y1 = -3e38f, z0 = 3e38f, z1 = -3e38f, hm = 0.f;
            if (lane < na) {
                x0 = x1 = sh.ax[lane]; y0 = y1 = sh.ay[lane]; z0 = z1 = sh.az[lane];
                hm = sh.aH[lane];
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
        unsigned long long grp_cands = 0;
        bool more_walk;
        do {
            __syncthreads();
            if (warp == 0) walk_batch<true>(sh.ws, a.nodes, a.node_hmax, L, FORCE_TILE, a.n_nodes);
            __syncthreads();
            const uint32_t total = sh.ws.total;
            more_walk = sh.ws.sp > 0;
            grp_cands += total;
            for (uint32_t tb = 0; tb < total; tb += FORCE_TILE) {
                float4 *tiles[3] = {t0, t1, t2};
                const float4 *srcs[3] = {a.xyzh, a.vc, a.raf};
                stage_tile<3>(sh.ws, tiles, srcs, tb, FORCE_TILE, L);
                __syncthreads();
                int tn = (int)min((uint32_t)FORCE_TILE, total - tb);
                if (sh.ws.pairwrap) force_units<KERNEL, true>(sh, t0, t1, t2, tn, L, a.alpha);
                else force_units<KERNEL, false>(sh, t0, t1, t2, tn, L, a.alpha);
                __syncthreads();
            }
        } while (more_walk);
        // a11: scatter to the caller's particle id
        if (tid < na) {
            uint32_t id = sh.aid[tid];
            a.acc[3 * (size_t)id] = (float)sh.fx[tid];
            a.acc[3 * (size_t)id + 1] = (float)sh.fy[tid];
            a.acc[3 * (size_t)id + 2] = (float)sh.fz[tid];
            a.dudt[id] = (float)sh.fdu[tid];
            a.vsig[id] = __int_as_float(sh.fvs[tid]);
        }
        if (warp == 0) {
            unsigned long long pr = (lane < na) ? (unsigned long long)(sh.aCnt[lane] - 1) : 0ull; // minus self
#pragma unroll
            for (int o = 16; o; o >>= 1) pr += __shfl_xor_sync(FULLMASK, pr, o);
            if (lane == 0) { st_pairs += pr; st_cands += grp_cands * (unsigned long long)na; }
        }
    }
    if (tid == 0) {
        if (st_cands) atomicAdd(&a.cnt->force_cands, st_cands);
        if (st_pairs) atomicAdd(&a.cnt->force_pairs, st_pairs);
    }
}

// gather the caller-order state into the sorted float4 arrays the gather streams through shared memory
__global__ void k_force_prep(int64_t n, const uint32_t *__restrict__ perm, const float4 *__restrict__ xyzm,
                             const float *__restrict__ vel, const float *__restrict__ u, const float *__restrict__ h,
                             const float *__restrict__ rho, const float *__restrict__ omega, float gamma,
                             float4 *__restrict__ xyzh, float4 *__restrict__ vc, float4 *__restrict__ raf)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t id = perm[i];
    float4 p = xyzm[i];
    float ui = u[id], ri = rho[id];
    float c = sqrtf(gamma * (gamma - 1.f) * ui);
    float A = (gamma - 1.f) * ui / (omega[id] * ri); // P/(Omega rho^2), P = (gamma-1) rho u
    xyzh[i] = make_float4(p.x, p.y, p.z, h[id]);
    vc[i] = make_float4(vel[3 * (int64_t)id], vel[3 * (int64_t)id + 1], vel[3 * (int64_t)id + 2], c);
    raf[i] = make_float4(ri, A, p.w, __uint_as_float((uint32_t)i));
}

// largest support radius inside every octree node: leaves scan their particles, then push the value
// up the parent chain with integer atomicMax (H > 0, so the float bit patterns order like integers)
__global__ void k_node_hmax(const SphCounters *cnt, const SphNode *__restrict__ nodes, const float4 *__restrict__ xyzh,
                            float *__restrict__ hmax)
{
    uint32_t nn = cnt->n_nodes;
    for (uint32_t nd = blockIdx.x * blockDim.x + threadIdx.x; nd < nn; nd += gridDim.x * blockDim.x) {
        SphNode p = nodes[nd];
        if (p.child != 0 || p.count == 0) continue;
        float m = 0.f;
        for (uint32_t s = 0; s < p.count; s++) m = fmaxf(m, xyzh[p.start + s].w);
        int mb = __float_as_int(m);
        uint32_t cur = nd;
        for (;;) {
            int old = atomicMax(reinterpret_cast<int *>(hmax) + cur, mb);
            if (cur == 0 || old >= mb) break;
            cur = nodes[cur].parent;
        }
    }
}

template <int KERNEL>
int launch(sph_ctx *ctx, const ForceArgs &a, int grid)
{
    size_t dyn = 3 * sizeof(float4) * FORCE_TILE;
    SPH_CUDA(ctx, cudaFuncSetAttribute(k_force<KERNEL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    k_force<KERNEL><<<grid, SPH_THREADS, dyn, ctx->stream>>>(a);
    SPH_CUDA(ctx, cudaGetLastError());
    return SPH_OK;
}

} // namespace

int sph_force_launch(sph_ctx *ctx, bool subset, int64_t n_items, const float *vel, const float *u, const float *h,
                     const float *rho, const float *omega, float *acc, float *dudt, float *vsig)
{
    cudaStream_t st = ctx->stream;
    const int64_t n = ctx->n;
    const int T = 256;
    cudaEventRecord(ctx->ev[4], st);
    k_force_prep<<<(int)((n + T - 1) / T), T, 0, st>>>(n, ctx->perm, ctx->xyzm, vel, u, h, rho, omega, ctx->prm.gamma,
                                                       ctx->f_xyzh, ctx->f_vc, ctx->f_raf);
    SPH_CUDA(ctx, cudaMemsetAsync(ctx->node_hmax, 0, sizeof(float) * ctx->n_nodes, st));
    k_node_hmax<<<ctx->device_sms * 4, 128, 0, st>>>(ctx->cnt, ctx->nodes, ctx->f_xyzh, ctx->node_hmax);
    sph_reset_counters(ctx, 1);
    ctx->launches += 3;
    cudaEventRecord(ctx->ev[5], st);
    ctx->ev_set[2] = true;

    ForceArgs a;
    a.nodes = ctx->nodes;
    a.n_nodes = (uint32_t)ctx->n_nodes;
    a.node_hmax = ctx->node_hmax;
    a.xyzh = ctx->f_xyzh; a.vc = ctx->f_vc; a.raf = ctx->f_raf;
    a.perm = ctx->perm;
    a.gstart = subset ? ctx->agrp_start : ctx->grp_start;
    a.n_groups = subset ? &ctx->cnt->n_agroups : &ctx->cnt->n_groups;
    a.item_slot = subset ? ctx->act_slot : nullptr;
    a.n_items = (uint32_t)n_items;
    a.cnt = ctx->cnt;
    a.L = ctx->prm.box;
    a.alpha = ctx->prm.alpha_visc;
    a.acc = acc; a.dudt = dudt; a.vsig = vsig;
    int64_t est_groups = subset ? n_items : ctx->n_groups;
    int grid = ctx->device_sms * 3;
    if (est_groups < grid) grid = (int)(est_groups > 0 ? est_groups : 1);
    cudaEventRecord(ctx->ev[6], st);
    int rc = ctx->prm.kernel == SPH_KERNEL_CUBIC ? launch<SPH_KERNEL_CUBIC>(ctx, a, grid) : launch<SPH_KERNEL_WC6>(ctx, a, grid);
    cudaEventRecord(ctx->ev[7], st);
    ctx->ev_set[3] = true;
    ctx->launches++;
    return rc;
}
