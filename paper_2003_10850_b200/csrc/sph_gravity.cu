// sph_gravity.cu -- SURVEY.md §8(f)-4: short-range Barnes-Hut gravity on the Morton-sorted particles, with the octree
// of the index build (cells from key prefixes) as the tree.
//
// The paper's gravity is a Barnes-Hut tree (plus a particle mesh for the long range) in which "particles interact
// with distant tree nodes as they were point-like pseudo particles" and the interaction is computed inside the walk
// branch, "which will limit the peak GPU performance" (PAPER.md:25 §1, :41, :102-104 §2.4).  Reading R23 of DESIGN.md:
// the short-range force of the TreePM split, Plummer softening, truncated at r_cut.  Here the walk is grouped -- one
// warp walks for a group of <= 32 neighbouring active particles and collects an interaction list of accepted nodes
// (monopoles: centre of mass, mass) and of leaf particle runs, which is then evaluated by all lanes -- so the pair
// arithmetic is separated from the walk branch.
#include <type_traits>

#include "sph_warp.cuh"

namespace {

#define GRAV_SEGS 96   // leaf runs per interaction-list batch (per warp)
#define GRAV_MONO 224  // accepted nodes per batch

struct GravArgs {
    const SphNode *nodes;
    const float4 *mom;      // per node: centre of mass, mass
    const float4 *xyzm;     // sorted particles
    const uint32_t *perm, *gstart;
    const unsigned int *n_groups;
    const uint32_t *item_slot;
    uint32_t n_items;
    SphCounters *cnt;
    float L, G, hrs, rcut, rcut2, eps2, theta2;  // hrs = 1 / (2 r_s)
    float *acc;
};

struct GravWarp {
    float4 mono[GRAV_MONO];
    uint32_t seg_start[GRAV_SEGS], seg_end[GRAV_SEGS];
    uint32_t stack[SPH_STK];
};

// G m_j * [erfc(r / 2 r_s) + r / (r_s sqrt(pi)) exp(-r^2 / 4 r_s^2)] / (r^2 + eps^2)^(3/2) for r < r_cut, else 0  (R23).
// With x = r / 2 r_s the bracket is exp(-x^2) * (P(t) + 2 x / sqrt(pi)), t = 1 / (1 + p x): erfc by the rational
// approximation 7.1.26 of Abramowitz & Stegun (|error| <= 1.5e-7, i.e. <= 1e-5 of the bracket at x = 2.25 where it is
// smallest), which shares the exponential with the second term -- one ex2, one rcp and six FMAs instead of erfcf + expf.
__device__ __forceinline__ float grav_pair(const GravArgs &a, float r2, float m)
{
    const float s2 = r2 + a.eps2;
    const float ri = rsqrt_ftz(fmaxf(s2, 1e-37f));
    const float r = r2 * rsqrt_ftz(fmaxf(r2, 1e-37f)), x = r * a.hrs;
    const float t = rcp_ftz(fmaf(0.3275911f, x, 1.f));
    const float P = t * fmaf(t, fmaf(t, fmaf(t, fmaf(t, 1.061405429f, -1.453152027f), 1.421413741f), -0.284496736f), 0.254829592f);
    const float fac = ex2_ftz(-1.4426950408889634f * x * x) * fmaf(1.1283791670955126f, x, P); // exp(-x^2), x <= r_cut / 2 r_s
    return r2 < a.rcut2 ? a.G * m * fac * ri * ri * ri : 0.f;
}

__global__ void __launch_bounds__(SPH_THREADS) k_gravity(GravArgs a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    GravWarp &W = reinterpret_cast<GravWarp *>(smem_raw)[warp];
    if (a.cnt->err | a.cnt->idx_err) return;
    const unsigned int n_groups = *a.n_groups;
    const float L = a.L;
    for (;;) {
        unsigned int grp = 0;
        if (lane == 0) grp = atomicAdd(&a.cnt->work, 1u);
        grp = __shfl_sync(FULLMASK, grp, 0);
        if (grp >= n_groups) break;
        const uint32_t i0 = a.gstart[grp];
        const uint32_t i1 = (grp + 1 < n_groups) ? a.gstart[grp + 1] : a.n_items;
        const int g = (int)(i1 - i0);
        const int f = 32 / g;
        const bool live = lane < g * f;
        const int ai = live ? lane % g : 0, s = live ? lane / g : 0;
        const uint32_t slot = a.item_slot ? a.item_slot[i0 + ai] : i0 + ai;
        const float4 pi = a.xyzm[slot];
        // the group's bounding box
        const float inf = __int_as_float(0x7f800000);
        const bool has = lane < g;
        const float x0 = warp_min(has ? pi.x : inf), x1 = warp_max(has ? pi.x : -inf);
        const float y0 = warp_min(has ? pi.y : inf), y1 = warp_max(has ? pi.y : -inf);
        const float z0 = warp_min(has ? pi.z : inf), z1 = warp_max(has ? pi.z : -inf);
        const float gcx = 0.5f * (x0 + x1), ghx = 0.5f * (x1 - x0) * (1.f + 1e-6f);
        const float gcy = 0.5f * (y0 + y1), ghy = 0.5f * (y1 - y0) * (1.f + 1e-6f);
        const float gcz = 0.5f * (z0 + z1), ghz = 0.5f * (z1 - z0) * (1.f + 1e-6f);
        const float rcw = a.rcut * (1.f + 1e-5f);
        const bool plain = x0 - rcw >= 0.f && x1 + rcw < L && y0 - rcw >= 0.f && y1 + rcw < L && z0 - rcw >= 0.f && z1 + rcw < L;
        double ax = 0.0, ay = 0.0, az = 0.0;
        int sp = 0;
        int nseg = 0, nmono = 0;
        __syncwarp();
        {
            const SphNode root = load_node(a.nodes, 0);
            if (root.child == 0) {
                if (root.count > 0 && lane == 0) { W.seg_start[0] = root.start; W.seg_end[0] = root.start + root.count; }
                nseg = root.count > 0 ? 1 : 0;
            } else {
                if (lane == 0) W.stack[0] = root.child;
                sp = 1;
            }
        }
        __syncwarp();
        while (sp > 0 || nseg > 0 || nmono > 0) {
            // walk: fill the interaction list
            while (sp > 0 && nseg <= GRAV_SEGS - 32 && nmono <= GRAV_MONO - 32) {
                const int npop = sp <= SPH_STK4 ? min(sp, 4) : 1;
                sp -= npop;
                const int e = lane >> 3;
                const bool valid = e < npop;
                const uint32_t idx = valid ? W.stack[sp + e] + (lane & 7) : 0u;
                const SphNode nd = load_node(a.nodes, idx);
                const float4 mo = __ldg(a.mom + idx);
                const float hh = nd.half * (1.f + 1e-6f) + 1e-6f * L;
                float dx = fabsf(gcx - nd.cx); dx = fminf(dx, L - dx); dx = fmaxf(dx - (ghx + hh), 0.f);
                float dy = fabsf(gcy - nd.cy); dy = fminf(dy, L - dy); dy = fmaxf(dy - (ghy + hh), 0.f);
                float dz = fabsf(gcz - nd.cz); dz = fminf(dz, L - dz); dz = fmaxf(dz - (ghz + hh), 0.f);
                const float rc = a.rcut * (1.f + 1e-5f);
                const bool pass = valid && nd.count > 0 && dx * dx + dy * dy + dz * dz <= rc * rc; // some point within r_cut
                // opening criterion: cell edge / distance from the group's box to the centre of mass < theta
                float cx = fabsf(gcx - mo.x); cx = fminf(cx, L - cx); cx = fmaxf(cx - ghx, 0.f);
                float cy = fabsf(gcy - mo.y); cy = fminf(cy, L - cy); cy = fmaxf(cy - ghy, 0.f);
                float cz = fabsf(gcz - mo.z); cz = fminf(cz, L - cz); cz = fmaxf(cz - ghz, 0.f);
                const float dc2 = cx * cx + cy * cy + cz * cz;
                const float l = 2.f * nd.half;
                const bool leaf = nd.child == 0;
                // (a cell the group touches is never accepted: dx = dy = dz = 0 means its particles may be arbitrarily close)
                const bool accept = pass && !leaf && l * l < a.theta2 * dc2 && (dx > 0.f || dy > 0.f || dz > 0.f);
                const bool emit = pass && leaf, push = pass && !leaf && !accept;
                const unsigned me = __ballot_sync(FULLMASK, emit), ma = __ballot_sync(FULLMASK, accept), mp = __ballot_sync(FULLMASK, push);
                if (emit) { const int p = nseg + __popc(me & lanemask_lt()); W.seg_start[p] = nd.start; W.seg_end[p] = nd.start + nd.count; }
                if (accept) W.mono[nmono + __popc(ma & lanemask_lt())] = mo;
                if (push) W.stack[sp + __popc(mp & lanemask_lt())] = nd.child;
                nseg += __popc(me); nmono += __popc(ma); sp += __popc(mp);
                __syncwarp();
            }
            auto evaluate = [&](auto plain_c) {
                constexpr bool PLAIN = decltype(plain_c)::value;
            // evaluate: lane = (active, stream); the streams split the accepted nodes and the flat sequence of the leaf
            // runs' particles; 16 terms at a time are summed in fp32, those sums in fp64
            if (live) {
                float bx = 0.f, by = 0.f, bz = 0.f;
                for (int i = s; i < nmono; i += f) {
                    const float4 q = W.mono[i];
                    const float ddx = (PLAIN ? pi.x - q.x : image_diff(pi.x, q.x, L)), ddy = (PLAIN ? pi.y - q.y : image_diff(pi.y, q.y, L)), ddz = (PLAIN ? pi.z - q.z : image_diff(pi.z, q.z, L));
                    const float t = grav_pair(a, fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx)), q.w);
                    bx = fmaf(-t, ddx, bx); by = fmaf(-t, ddy, by); bz = fmaf(-t, ddz, bz);
                }
                ax += (double)bx; ay += (double)by; az += (double)bz;
                bx = by = bz = 0.f;
                if (nseg > 0) {
                    int k = 0, since = 0;
                    uint32_t j = W.seg_start[0] + (uint32_t)s, e = W.seg_end[0];
                    for (;;) {
                        while (j >= e && ++k < nseg) { // step over the ends of the runs
                            j = W.seg_start[k] + (j - e);
                            e = W.seg_end[k];
                        }
                        if (k >= nseg) break;
                        const float4 q = __ldg(a.xyzm + j);
                        const float ddx = (PLAIN ? pi.x - q.x : image_diff(pi.x, q.x, L)), ddy = (PLAIN ? pi.y - q.y : image_diff(pi.y, q.y, L)), ddz = (PLAIN ? pi.z - q.z : image_diff(pi.z, q.z, L));
                        const float t = j != slot ? grav_pair(a, fmaf(ddz, ddz, fmaf(ddy, ddy, ddx * ddx)), q.w) : 0.f;
                        bx = fmaf(-t, ddx, bx); by = fmaf(-t, ddy, by); bz = fmaf(-t, ddz, bz);
                        j += (uint32_t)f;
                        if (++since == 16) { // (fp32 partial sums stay short: DESIGN.md R15's argument for the force pass)
                            ax += (double)bx; ay += (double)by; az += (double)bz;
                            bx = by = bz = 0.f;
                            since = 0;
                        }
                    }
                }
                ax += (double)bx; ay += (double)by; az += (double)bz;
            }
            };
            // no wall within r_cut of the group: every pair closer than r_cut has its nearest image at the plain difference,
            // and a plain difference is never shorter than the nearest-image one (pairs beyond r_cut contribute nothing)
            if (plain) evaluate(std::true_type());
            else evaluate(std::false_type());
            nseg = nmono = 0;
            __syncwarp();
        }
        // cross-stream totals, scatter to the caller's id
        for (int d = 1; d < f; d <<= 1) {
            const bool take = live && s + d < f;
            const int from = take ? lane + g * d : lane;
            const double tx = __shfl_sync(FULLMASK, ax, from), ty = __shfl_sync(FULLMASK, ay, from), tz = __shfl_sync(FULLMASK, az, from);
            if (take) { ax += tx; ay += ty; az += tz; }
        }
        if (lane < g) {
            const uint32_t id = a.perm[slot];
            a.acc[3 * (size_t)id] = (float)ax;
            a.acc[3 * (size_t)id + 1] = (float)ay;
            a.acc[3 * (size_t)id + 2] = (float)az;
        }
    }
}

// mass and centre of mass of the nodes of one octree level (children first: launched from the deepest level up)
__global__ void k_node_moments(const SphCounters *cnt, int level, const SphNode *__restrict__ nodes, const float4 *__restrict__ xyzm,
                               float4 *__restrict__ mom)
{
    const uint32_t beg = cnt->lvl_begin[level], end = min(cnt->lvl_begin[level + 1], cnt->n_nodes);
    for (uint32_t nd = beg + blockIdx.x * blockDim.x + threadIdx.x; nd < end; nd += gridDim.x * blockDim.x) {
        const SphNode p = nodes[nd];
        double m = 0.0, x = 0.0, y = 0.0, z = 0.0;
        if (p.child == 0) {
            for (uint32_t s = 0; s < p.count; s++) {
                const float4 q = xyzm[p.start + s];
                m += q.w; x += (double)q.w * q.x; y += (double)q.w * q.y; z += (double)q.w * q.z;
            }
        } else {
            for (int c = 0; c < 8; c++) {
                const float4 q = mom[p.child + c];
                m += q.w; x += (double)q.w * q.x; y += (double)q.w * q.y; z += (double)q.w * q.z;
            }
        }
        mom[nd] = m > 0.0 ? make_float4((float)(x / m), (float)(y / m), (float)(z / m), (float)m) : make_float4(p.cx, p.cy, p.cz, 0.f);
    }
}

} // namespace

int sph_gravity_launch(sph_ctx *ctx, bool subset, int64_t n_items, float G, float r_s, float r_cut, float eps, float theta, float *acc)
{
    cudaStream_t st = ctx->stream;
    if (!ctx->node_mom || ctx->node_mom_cap < ctx->node_cap) {
        if (ctx->node_mom) cudaFree(ctx->node_mom);
        ctx->node_mom = nullptr;
        ctx->node_mom_cap = 0;
        SPH_CUDA(ctx, cudaMalloc((void **)&ctx->node_mom, sizeof(float4) * (size_t)ctx->node_cap));
        ctx->node_mom_cap = ctx->node_cap;
    }
    for (int level = SPH_LMAX; level >= 0; level--)
        k_node_moments<<<level < 3 ? 1 : ctx->device_sms * 2, 128, 0, st>>>(ctx->cnt, level, ctx->nodes, ctx->xyzm, ctx->node_mom);
    sph_reset_counters(ctx, 1, subset);
    GravArgs a;
    a.nodes = ctx->nodes; a.mom = ctx->node_mom; a.xyzm = ctx->xyzm; a.perm = ctx->perm;
    a.gstart = subset ? ctx->agrp_start : ctx->grp_start;
    a.n_groups = subset ? &ctx->cnt->n_agroups : &ctx->cnt->n_groups;
    a.item_slot = subset ? ctx->act_slot : nullptr;
    a.n_items = (uint32_t)n_items;
    a.cnt = ctx->cnt;
    a.L = ctx->prm.box; a.G = G; a.hrs = 0.5f / r_s; a.rcut = r_cut; a.rcut2 = r_cut * r_cut; a.eps2 = eps * eps; a.theta2 = theta * theta;
    a.acc = acc;
    const size_t dyn = sizeof(GravWarp) * SPH_WARPS;
    SPH_CUDA(ctx, cudaFuncSetAttribute(k_gravity, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    int per_sm = 1;
    SPH_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_gravity, SPH_THREADS, dyn));
    if (per_sm < 1) return sph_fail(ctx, SPH_E_INTERNAL, "k_gravity does not fit on an SM");
    int64_t grid = (int64_t)ctx->device_sms * per_sm;
    const int64_t need = (n_items + SPH_WARPS - 1) / SPH_WARPS;
    if (need < grid) grid = need > 0 ? need : 1;
    k_gravity<<<(int)grid, SPH_THREADS, dyn, st>>>(a);
    ctx->launches += SPH_LMAX + 3;
    SPH_CUDA(ctx, cudaGetLastError());
    return SPH_OK;
}
