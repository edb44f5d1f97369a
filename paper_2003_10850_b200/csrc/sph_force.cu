// sph_force.cu -- steps a5, a6, a10, a11: symmetric hydro-force pair sum (pressure gradient +
// signal-velocity artificial viscosity) and the maximum signal velocity, for the active particles.
//
// "the second one computes hydrodynamic forces" (§1); same search pattern as the density
// module (§1).  Formulas: DESIGN.md readings R8-R12.  The neighbour set is symmetric,
// r_ij < max(H_i, H_j) (R10): the walk prunes a node only if it is farther from the group than both
// the group's reach and the largest support radius inside the node.
//
// Same CTA-per-group mapping as sph_density.cu: thread = (active, stream).  The candidate runs found by
// the walk are staged tile by tile in shared memory, each candidate twice: component arrays X[], Y[],
// Z[], H2[] for the packed distance tests, and three 16-byte records (x,y,z,slot | v,c | rho,A,m,1/H) for
// the hit evaluation.  A hit pushes the candidate's tile-local index onto the thread's queue; queued
// hits are evaluated in bulk from shared memory (no global access per hit); a, du/dt are accumulated
// in fp64 per thread (R15).
#include "sph_warp.cuh"

namespace {

struct ForceArgs {
    const SphNode *nodes;
    const float *node_hmax;
    const float4 *xyzh, *vc; // sorted: (x,y,z,H); 32-byte records (vx,vy,vz,c | rho, A, m, 1/H) at vc[2j], vc[2j+1]
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
// w'(q) for the two arguments of a pair, (r / H_i, r / H_j), in one packed f32x2 chain
template <int KERNEL>
__device__ __forceinline__ float2 kern_dw2(float2 q)
{
    const float2 one = make_float2(1.f, 1.f);
    float2 t = __ffma2_rn(q, make_float2(-1.f, -1.f), one);
    t = make_float2(fmaxf(t.x, 0.f), fmaxf(t.y, 0.f));
    const float2 t2 = __fmul2_rn(t, t);
    if (KERNEL == SPH_KERNEL_CUBIC) {
        const float2 a = __fmul2_rn(q, __ffma2_rn(make_float2(18.f, 18.f), q, make_float2(-12.f, -12.f)));
        const float2 b = __fmul2_rn(make_float2(-6.f, -6.f), t2);
        return make_float2(q.x <= 0.5f ? a.x : b.x, q.y <= 0.5f ? a.y : b.y);
    } else {
        const float2 t4 = __fmul2_rn(t2, t2), t7 = __fmul2_rn(__fmul2_rn(t4, t2), t);
        const float2 p = __ffma2_rn(q, __ffma2_rn(make_float2(16.f, 16.f), q, make_float2(7.f, 7.f)), one);
        return __fmul2_rn(__fmul2_rn(__fmul2_rn(make_float2(-22.f, -22.f), q), t7), p);
    }
}
template <int KERNEL>
__device__ __forceinline__ float kern_sigma()
{
    return KERNEL == SPH_KERNEL_CUBIC ? 2.54647908947032537f : 6.78895304126365994f;
}

struct ForceCta {
    // one tile of candidates in the batch's frame: component arrays for the tests (NaN-padded like the
    // density kernel's) and the state records for the hits
    alignas(16) float X[SPH_FTILE + 8];
    alignas(16) float Y[SPH_FTILE + 8];
    alignas(16) float Z[SPH_FTILE + 8];
    alignas(16) float H2[SPH_FTILE + 8];
    alignas(16) float4 r0[SPH_FTILE]; // x, y, z (frame), sorted slot (bits)
    alignas(16) float4 r1[SPH_FTILE]; // vx, vy, vz, c
    alignas(16) float4 r2[SPH_FTILE]; // rho, A, m, 1/H
    alignas(16) uint16_t q[SPH_QCAP_FORCE * SPH_THREADS]; // hit queues: entry k of thread t at [k * SPH_THREADS + t]
    WalkShared W;
    unsigned int gnext;
};

#define SPH_FQSTRIDE (2u * SPH_THREADS) // bytes between consecutive queue entries of a thread

// per-thread state of the thread's active and its running sums
struct ForceLane {
    float xi, yi, zi, h2, hinv, f4;  // position, H^2, 1/H, sigma/H^4
    float xf, yf, zf;                // position in the batch's frame
    float vx, vy, vz, c, rho, A;
    uint32_t slot;
    double px, py, pz, pdu;          // fp64 accumulators (R15: "fp64 accumulation where needed")
    float pvs;
    int cn, cnt;                     // hits evaluated; hits queued
};

__device__ __forceinline__ void sts_u16(uint32_t addr, uint32_t v)
{
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v)); // no memory clobber: see sts_f32
}
__device__ __forceinline__ uint32_t lds_u16(uint32_t addr)
{
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr) : "memory");
    return (uint32_t)v;
}

// evaluate the m newest queued hits of every thread of the warp (n = warp-wide maximum of m) from the
// tile's state records
template <int KERNEL, bool PAIRWRAP>
__device__ __forceinline__ void drain(const ForceCta &C, const ForceArgs &a, uint32_t q0, ForceLane &A, int n)
{
    const int m = min(n, A.cnt), base = A.cnt - m;
    const float L = a.L, alpha = a.alpha;
    uint32_t ra = q0 + (uint32_t)base * SPH_FQSTRIDE;
#pragma unroll 2
    for (int k = 0; k < n; k++, ra += SPH_FQSTRIDE) {
        if (k < m) {
            const uint32_t j = lds_u16(ra);
            const float4 P0 = C.r0[j], P1 = C.r1[j], P2 = C.r2[j];
            float dx, dy, dz;
            if (PAIRWRAP) {
                dx = image_diff(A.xi, P0.x, L); dy = image_diff(A.yi, P0.y, L); dz = image_diff(A.zi, P0.z, L);
            } else {
                dx = A.xf - P0.x; dy = A.yf - P0.y; dz = A.zf - P0.z;
            }
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            const float rinv = rsqrtf(fmaxf(r2, 1e-37f));
            const float r = r2 * rinv;
            const float hinv_j = P2.w; // 1 / H_j, correctly rounded once per particle (k_force_prep)
            const float hj2 = hinv_j * hinv_j;
            const float2 dw = kern_dw2<KERNEL>(__fmul2_rn(make_float2(r, r), make_float2(A.hinv, hinv_j)));
            const float Fi = A.f4 * dw.x;
            const float Fj = kern_sigma<KERNEL>() * hj2 * hj2 * dw.y;
            const float dvx = A.vx - P1.x, dvy = A.vy - P1.y, dvz = A.vz - P1.z;
            const float vr = fmaf(dvz, dz, fmaf(dvy, dy, dvx * dx)) * rinv;
            const float mu = fminf(vr, 0.f);
            const float vs = A.c + P1.w - 3.f * mu;
            const float Pi = -alpha * vs * mu * __fdividef(1.f, A.rho + P2.x);
            const float Fbar = 0.5f * (Fi + Fj);
            const float AiFi = A.A * Fi;
            const float pv = Pi * Fbar;
            const bool other = __float_as_uint(P0.w) != A.slot; // j == i: no self force, no self signal velocity
            // select, not multiply by zero: a lone particle has Omega = 0, hence A = inf
            const float tr = other ? P2.z * (AiFi + fmaf(P2.y, Fj, pv)) * rinv : 0.f;
            const float du = other ? P2.z * fmaf(0.5f, pv, AiFi) * vr : 0.f;
            A.px -= (double)(tr * dx);
            A.py -= (double)(tr * dy);
            A.pz -= (double)(tr * dz);
            A.pdu += (double)du;
            A.pvs = fmaxf(A.pvs, other ? vs : 0.f);
        }
    }
    A.cn += m;
    A.cnt = base;
}

// one candidate against this thread's active (symmetric set, R10): hit if r^2 < max(H_i, H_j)^2
__device__ __forceinline__ void push_if(const ForceLane &A, uint32_t &qw, float r2, float hj2, uint32_t idx)
{
    if (r2 < fmaxf(A.h2, hj2)) {
        sts_u16(qw, idx);
        qw += SPH_FQSTRIDE;
    }
}

// Test the nq candidate quads of the staged tile against this thread's active; a hit pushes the
// candidate's tile-local index onto the thread's queue.
template <int KERNEL, bool PAIRWRAP>
__device__ __forceinline__ void consume(const ForceCta &C, const ForceArgs &a, uint32_t q0, ForceLane &A, int nq, int s, int f,
                                        bool live)
{
    const float4 *X4 = reinterpret_cast<const float4 *>(C.X), *Y4 = reinterpret_cast<const float4 *>(C.Y);
    const float4 *Z4 = reinterpret_cast<const float4 *>(C.Z), *H4 = reinterpret_cast<const float4 *>(C.H2);
    const float L = a.L;
    const float2 nx = make_float2(-A.xf, -A.xf), ny = make_float2(-A.yf, -A.yf), nz = make_float2(-A.zf, -A.zf);
    const int steps = (nq + f - 1) / f; // CTA-uniform
    int qd = s;
    for (int t0 = 0; t0 < steps; t0 += SPH_QSTEP_FORCE) {
        const int nt = min(SPH_QSTEP_FORCE, steps - t0);
        const int mx = __reduce_max_sync(FULLMASK, A.cnt);
        if (mx + 4 * nt > SPH_QCAP_FORCE) {
            const int mn = __reduce_min_sync(FULLMASK, live ? A.cnt : 0x7fffffff);
            drain<KERNEL, PAIRWRAP>(C, a, q0, A, max(min(mn, mx), mx + 4 * nt - SPH_QCAP_FORCE));
        }
        uint32_t qw = q0 + (uint32_t)A.cnt * SPH_FQSTRIDE;
#pragma unroll 2
        for (int t = 0; t < nt; t++) {
            const int qi = min(qd, nq);
            qd += f;
            const float4 x = X4[qi], y = Y4[qi], z = Z4[qi], h = H4[qi]; // h: H_j^2 (squared once per candidate by the gather)
            float2 ra, rb;
            if (PAIRWRAP) {
                const float dx0 = image_diff(A.xi, x.x, L), dx1 = image_diff(A.xi, x.y, L);
                const float dx2 = image_diff(A.xi, x.z, L), dx3 = image_diff(A.xi, x.w, L);
                const float dy0 = image_diff(A.yi, y.x, L), dy1 = image_diff(A.yi, y.y, L);
                const float dy2 = image_diff(A.yi, y.z, L), dy3 = image_diff(A.yi, y.w, L);
                const float dz0 = image_diff(A.zi, z.x, L), dz1 = image_diff(A.zi, z.y, L);
                const float dz2 = image_diff(A.zi, z.z, L), dz3 = image_diff(A.zi, z.w, L);
                ra = make_float2(fmaf(dz0, dz0, fmaf(dy0, dy0, dx0 * dx0)), fmaf(dz1, dz1, fmaf(dy1, dy1, dx1 * dx1)));
                rb = make_float2(fmaf(dz2, dz2, fmaf(dy2, dy2, dx2 * dx2)), fmaf(dz3, dz3, fmaf(dy3, dy3, dx3 * dx3)));
            } else {
                const float2 dxa = __fadd2_rn(make_float2(x.x, x.y), nx), dxb = __fadd2_rn(make_float2(x.z, x.w), nx);
                const float2 dya = __fadd2_rn(make_float2(y.x, y.y), ny), dyb = __fadd2_rn(make_float2(y.z, y.w), ny);
                const float2 dza = __fadd2_rn(make_float2(z.x, z.y), nz), dzb = __fadd2_rn(make_float2(z.z, z.w), nz);
                ra = __ffma2_rn(dza, dza, __ffma2_rn(dya, dya, __fmul2_rn(dxa, dxa)));
                rb = __ffma2_rn(dzb, dzb, __ffma2_rn(dyb, dyb, __fmul2_rn(dxb, dxb)));
            }
            const uint32_t i0 = 4u * (uint32_t)qi;
            push_if(A, qw, ra.x, h.x, i0);
            push_if(A, qw, ra.y, h.y, i0 + 1u);
            push_if(A, qw, rb.x, h.z, i0 + 2u);
            push_if(A, qw, rb.y, h.w, i0 + 3u);
        }
        A.cnt = (int)((qw - q0) / SPH_FQSTRIDE);
    }
}

// Stage tile t of the nt tiles of a walk batch: test arrays + state records.  The batch's candidates are
// dealt onto the tiles one by one, round-robin (flat position p goes to tile p % nt, slot p / nt): every
// tile is a uniform, fine-grained sample of the whole candidate set, so every thread finds its fair share
// of hits in every tile and the bulk evaluation at the end of a tile keeps the lanes busy (a tile of
// consecutive candidates is a compact region, near some actives and out of reach of the rest).
// Returns the number of candidates of the tile (slots [0, cnt) are in use).
__device__ __forceinline__ uint32_t gather_tile(ForceCta &C, const WalkCtl &ctl, uint32_t t, uint32_t nt, const ForceArgs &a)
{
    const int tid = threadIdx.x;
    const float L = a.L;
    const WalkShared &W = C.W;
    const bool rec = !ctl.pairwrap && (ctl.thx < 1e30f || ctl.thy < 1e30f || ctl.thz < 1e30f); // CTA-uniform
    const uint32_t cnt = (ctl.total - t + nt - 1u) / nt; // t < nt <= total
    for (uint32_t sl = tid; sl < cnt; sl += SPH_THREADS) {
        const uint32_t p = sl * nt + t;
        const int k = seg_of(W, ctl.n_seg, p);
        const uint32_t j = W.seg_start[k] + (p - W.seg_pre[k]);
        float4 c = ldg_nc(a.xyzh + j);
        const float4 v = ldg_nc(a.vc + 2 * (size_t)j), w = ldg_nc(a.vc + 2 * (size_t)j + 1);
        if (rec) { c.x = recentre(c.x, ctl.thx, L); c.y = recentre(c.y, ctl.thy, L); c.z = recentre(c.z, ctl.thz, L); }
        C.X[sl] = c.x; C.Y[sl] = c.y; C.Z[sl] = c.z; C.H2[sl] = c.w * c.w;
        C.r0[sl] = make_float4(c.x, c.y, c.z, __uint_as_float(j));
        C.r1[sl] = v;
        C.r2[sl] = w;
    }
    const uint32_t nq = (cnt + 3u) >> 2;
    for (uint32_t o = cnt + tid; o < 4u * nq + 4u; o += SPH_THREADS) { C.X[o] = SPH_NANF; C.Y[o] = 0.f; C.Z[o] = 0.f; C.H2[o] = 0.f; }
    return cnt;
}

template <int KERNEL>
__global__ void __launch_bounds__(SPH_THREADS, SPH_CTAS_FORCE) k_force(ForceArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    ForceCta &C = *reinterpret_cast<ForceCta *>(smem_raw);
    const float L = a.L;
    if (a.cnt->bad_ids) return; // an active id was out of range: compute nothing (uniform over the grid)
    const unsigned int n_groups = *a.n_groups;
    unsigned long long st_cands = 0, st_pairs = 0, st_staged = 0; // thread 0 / warp 0
    const uint32_t q0 = smem_u32(C.q + tid);

    for (;;) {
        __syncthreads(); // the previous group's shared state is dead
        if (tid == 0) C.gnext = atomicAdd(&a.cnt->work, 1u);
        __syncthreads();
        const unsigned int grp = C.gnext;
        if (grp >= n_groups) break;
        const uint32_t i0 = a.gstart[grp];
        const uint32_t i1 = (grp + 1 < n_groups) ? a.gstart[grp + 1] : a.n_items;
        const int g = (int)(i1 - i0);
        SPH_ASSERT(g >= 1 && g <= SPH_MAXB);
        const int f = streams_for(g);
        const bool live = tid < g * f;
        const int ai = live ? tid % g : 0, s = live ? tid / g : 0;
        ForceLane A;
        const uint32_t slot = a.item_slot ? a.item_slot[i0 + ai] : i0 + ai;
        const float4 p0 = a.xyzh[slot], p1 = a.vc[2 * (size_t)slot], p2 = a.vc[2 * (size_t)slot + 1];
        A.slot = slot;
        A.xi = live ? p0.x : SPH_NANF; // dead threads never hit
        A.yi = p0.y; A.zi = p0.z;
        A.h2 = p0.w * p0.w;
        A.hinv = 1.f / p0.w;
        const float h2i = A.hinv * A.hinv;
        A.f4 = kern_sigma<KERNEL>() * h2i * h2i;
        A.vx = p1.x; A.vy = p1.y; A.vz = p1.z; A.c = p1.w;
        A.rho = p2.x; A.A = p2.y;
        A.px = A.py = A.pz = A.pdu = 0.0;
        A.pvs = 0.f;
        A.cn = A.cnt = 0;
        // warp 0 (thread i < g holds active i): bounding box and reach of the group
        if (warp == 0) publish_box(C.W, lane < g, p0.x, p0.y, p0.z, warp_max(lane < g ? p0.w : 0.f));
        __syncthreads();
        walk_cta<true>(C.W, a.nodes, a.node_hmax, L, true);
        unsigned long long cands = 0;
        for (;;) {
            const WalkCtl ctl = walk_result(C.W);
            cands += ctl.total;
            A.xf = ctl.pairwrap ? A.xi : recentre(A.xi, ctl.thx, L);
            A.yf = ctl.pairwrap ? A.yi : recentre(A.yi, ctl.thy, L);
            A.zf = ctl.pairwrap ? A.zi : recentre(A.zi, ctl.thz, L);
            const uint32_t nt = (ctl.total + SPH_FTILE - 1) / SPH_FTILE;
            for (uint32_t c = 0; c < nt; c++) {
                const uint32_t cnt = gather_tile(C, ctl, c, nt, a);
                st_staged += cnt;
                __syncthreads();
                const int nq = (int)((cnt + 3u) >> 2);
                // queued hits refer to this tile's records: all of them are evaluated before the tile is replaced
                if (ctl.pairwrap) {
                    consume<KERNEL, true>(C, a, q0, A, nq, s, f, live);
                    drain<KERNEL, true>(C, a, q0, A, __reduce_max_sync(FULLMASK, A.cnt));
                } else {
                    consume<KERNEL, false>(C, a, q0, A, nq, s, f, live);
                    drain<KERNEL, false>(C, a, q0, A, __reduce_max_sync(FULLMASK, A.cnt));
                }
                __syncthreads();
            }
            if (ctl.sp <= 0) break;
            walk_cta<true>(C.W, a.nodes, a.node_hmax, L, false);
        }
        // cross-stream totals through shared memory (the tile is dead): fp64, ascending stream order
        double *pX = reinterpret_cast<double *>(C.r0), *pY = pX + SPH_THREADS, *pZ = pY + SPH_THREADS, *pU = pZ + SPH_THREADS;
        float *pV = reinterpret_cast<float *>(pU + SPH_THREADS);
        int *pn = reinterpret_cast<int *>(pV + SPH_THREADS);
        pX[tid] = A.px; pY[tid] = A.py; pZ[tid] = A.pz; pU[tid] = A.pdu; pV[tid] = A.pvs; pn[tid] = A.cn;
        __syncthreads();
        if (warp == 0) {
            double X = 0.0, Y = 0.0, Z = 0.0, U = 0.0;
            float V = 0.f;
            int cn = 0;
            if (lane < g) {
                for (int t = lane; t < g * f; t += g) {
                    X += pX[t]; Y += pY[t]; Z += pZ[t]; U += pU[t]; V = fmaxf(V, pV[t]); cn += pn[t];
                }
                // a11: scatter to the caller's particle id
                const uint32_t id = a.perm[slot];
                a.acc[3 * (size_t)id] = (float)X;
                a.acc[3 * (size_t)id + 1] = (float)Y;
                a.acc[3 * (size_t)id + 2] = (float)Z;
                a.dudt[id] = (float)U;
                a.vsig[id] = V;
            }
            unsigned long long pr = (lane < g) ? (unsigned long long)(cn - 1) : 0ull; // minus self
#pragma unroll
            for (int o = 16; o; o >>= 1) pr += __shfl_xor_sync(FULLMASK, pr, o);
            st_pairs += pr;
            st_cands += cands * (unsigned long long)g;
        }
    }
    if (tid == 0) {
        if (st_cands) atomicAdd(&a.cnt->force_cands, st_cands);
        if (st_pairs) atomicAdd(&a.cnt->force_pairs, st_pairs);
        atomicAdd(&a.cnt->force_staged, st_staged);
    }
}

// gather the caller-order state into the sorted float4 arrays the gather streams through shared memory
__global__ void k_force_prep(int64_t n, const uint32_t *__restrict__ perm, const float4 *__restrict__ xyzm,
                             const float *__restrict__ vel, const float *__restrict__ u, const float *__restrict__ h,
                             const float *__restrict__ rho, const float *__restrict__ omega, float gamma,
                             float4 *__restrict__ xyzh, float4 *__restrict__ vc)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t id = perm[i];
    float4 p = xyzm[i];
    float ui = u[id], ri = rho[id];
    float c = sqrtf(gamma * (gamma - 1.f) * ui);
    float A = (gamma - 1.f) * ui / (omega[id] * ri); // P/(Omega rho^2), P = (gamma-1) rho u
    xyzh[i] = make_float4(p.x, p.y, p.z, h[id]);
    vc[2 * i] = make_float4(vel[3 * (int64_t)id], vel[3 * (int64_t)id + 1], vel[3 * (int64_t)id + 2], c);
    vc[2 * i + 1] = make_float4(ri, A, p.w, 1.f / h[id]);
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
int launch(sph_ctx *ctx, const ForceArgs &a, int64_t est_groups)
{
    size_t dyn = sizeof(ForceCta);
    auto kfn = k_force<KERNEL>;
    SPH_CUDA(ctx, cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    int per_sm = 1;
    SPH_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kfn, SPH_THREADS, dyn));
    if (per_sm < 1) return sph_fail(ctx, SPH_E_INTERNAL, "k_force does not fit on an SM");
    int64_t grid = (int64_t)ctx->device_sms * per_sm;
    if (est_groups < grid) grid = est_groups > 0 ? est_groups : 1;
    kfn<<<(int)grid, SPH_THREADS, dyn, ctx->stream>>>(a);
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
                                                       ctx->f_xyzh, ctx->f_vc);
    SPH_CUDA(ctx, cudaMemsetAsync(ctx->node_hmax, 0, sizeof(float) * ctx->n_nodes, st));
    k_node_hmax<<<ctx->device_sms * 4, 128, 0, st>>>(ctx->cnt, ctx->nodes, ctx->f_xyzh, ctx->node_hmax);
    sph_reset_counters(ctx, 1, subset);
    ctx->launches += 3;
    cudaEventRecord(ctx->ev[5], st);
    ctx->ev_set[2] = true;

    ForceArgs a;
    a.nodes = ctx->nodes;
    a.node_hmax = ctx->node_hmax;
    a.xyzh = ctx->f_xyzh; a.vc = ctx->f_vc;
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
    cudaEventRecord(ctx->ev[6], st);
    int rc = ctx->prm.kernel == SPH_KERNEL_CUBIC ? launch<SPH_KERNEL_CUBIC>(ctx, a, est_groups) : launch<SPH_KERNEL_WC6>(ctx, a, est_groups);
    cudaEventRecord(ctx->ev[7], st);
    ctx->ev_set[3] = true;
    ctx->launches++;
    return rc;
}
