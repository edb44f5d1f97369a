// sph_force.cu -- steps a5, a6, a10, a11: symmetric hydro-force pair sum (pressure gradient +
// signal-velocity artificial viscosity) and the maximum signal velocity, for the active particles.
//
// "the second one computes hydrodynamic forces" (§1); same search pattern as the density
// module (§1).  Formulas: DESIGN.md readings R8-R12.  The neighbour set is symmetric,
// r_ij < max(H_i, H_j) (R10): the walk prunes a node only if it is farther from the group than both
// the group's reach and the largest support radius inside the node.
//
// Same warp-per-group mapping as sph_density.cu: lane = (active, stream); candidates' (x,y,z,H) are
// gathered chunk by chunk into the warp's shared-memory slot and tested; a hit pushes the candidate's sorted slot
// onto the lane's queue; queued hits are evaluated in bulk, fetching the pair's remaining state
// (velocity, sound speed, rho, A, m) from the sorted arrays through L1.
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
    // improved-SPH extension (MODE_IMPROVED, MODE_GRADV; R17-R20)
    const float4 *ext;                 // sorted: (alpha, shear limiter f, u, -) per particle; MODE_CONDUCT: (kappa, T = u, -, -)
    float gm1;                         // gamma - 1
    float alpha_cond, alpha_min, alpha_max, decay_l;
    float *dalpha;                     // d alpha / dt of the active particles
    float *divv, *curlv;               // MODE_GRADV outputs
};

// pair physics of the gather kernel: the base hydro force (R8-R12), the same with the improved-SPH terms
// (per-particle alpha, shear limiter, artificial conduction: R18-R20), the velocity-gradient sums (R17), or the
// thermal-conduction pair sum (R21)
enum { MODE_BASE = SPH_MODE_BASE, MODE_IMPROVED = SPH_MODE_IMPROVED, MODE_GRADV = SPH_MODE_GRADV, MODE_CONDUCT = SPH_MODE_CONDUCT };

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

struct ForceWarp {
    float4 slot[SPH_CH];                // one chunk of candidates as pair records (x,y,z,H)
    WarpWalk ws;
    uint32_t q[SPH_QCAP_FORCE * 32];          // hit queue: sorted slot of the neighbour
    alignas(16) uint32_t gidx[SPH_CH];              // sorted slot of every candidate of the chunk
};

// per-lane state of the lane's active and its running sums
struct ForceLane {
    float xi, yi, zi, h2, hinv, f4;  // position, H^2, 1/H, sigma/H^4
    float vx, vy, vz, c, rho, A;
    float al, fb, u, P;     // MODE_IMPROVED: alpha_i, limiter f_i, u_i, P_i
    uint32_t slot;
    double px, py, pz, pdu; // fp64 accumulators of a and du/dt (R15: "fp64 accumulation where needed");
                            // MODE_GRADV: of the curl (3) and the divergence sums
    float pvs;
    int cn, cnt;
};

// frame of the batch the queued hits were found in (see walk_batch)
struct Frame {
    float thx, thy, thz;
    bool pairwrap;
    bool rec; // some axis is recentred (thr finite); false: raw coordinates are already the frame
};

// evaluate the m newest queued hits of every lane (n = warp-wide maximum of m)
// WRAP: 0 raw coordinate differences, 1 recentred frame, 2 per-pair nearest image
template <int KERNEL, int WRAP, int MODE>
__device__ __forceinline__ void drain(const ForceArgs &a, uint32_t q0, ForceLane &A, int n, const Frame &fr)
{
    const int m = min(n, A.cnt), base = A.cnt - m;
    const float L = a.L, alpha = a.alpha;
    const float xf = WRAP == 1 ? recentre(A.xi, fr.thx, L) : A.xi;
    const float yf = WRAP == 1 ? recentre(A.yi, fr.thy, L) : A.yi;
    const float zf = WRAP == 1 ? recentre(A.zi, fr.thz, L) : A.zi;
    // the hits of one call (at most a queue's worth: 32) are summed in fp32, the calls in fp64: the accumulators of
    // R15 stay out of the inner loop's registers at no measurable cost in accuracy
    float sx = 0.f, sy = 0.f, sz = 0.f, su = 0.f;
    uint32_t qa = q0 + (uint32_t)base * 128u; // shared-memory address of the next queued hit (q0: the lane's entry 0)
#pragma unroll 2
    for (int k = 0; k < n; k++) {
        if (k < m) {
            const uint32_t j = lds_u32(qa); // (volatile: ordered after the pushes)
            qa += 128u;
            const float4 P0 = __ldg(a.xyzh + j), P1 = __ldg(a.vc + 2 * (size_t)j), P2 = __ldg(a.vc + 2 * (size_t)j + 1);
            float dx, dy, dz;
            if (WRAP == 2) {
                dx = image_diff(A.xi, P0.x, L); dy = image_diff(A.yi, P0.y, L); dz = image_diff(A.zi, P0.z, L);
            } else if (WRAP == 1) {
                dx = xf - recentre(P0.x, fr.thx, L); dy = yf - recentre(P0.y, fr.thy, L); dz = zf - recentre(P0.z, fr.thz, L);
            } else {
                dx = xf - P0.x; dy = yf - P0.y; dz = zf - P0.z;
            }
            const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            // 1/r to ~1 ulp: the hardware approximation (2 ulp) plus one Newton step.  The pair term's error is
            // dominated by the error of r amplified by w''/w' (~10), and a sum of ~500 such terms is compared
            // with 1e-7 of the sum of their magnitudes (R15)
            const float r2c = fmaxf(r2, 1e-37f);
            float rinv = rsqrt_ftz(r2c);
            rinv = rinv * fmaf(-0.5f * r2c, rinv * rinv, 1.5f);
            const float r = r2 * rinv;
            const bool other = j != A.slot; // j == i: no self force, no self signal velocity
            if (MODE == MODE_GRADV) {
                // R17: m_j dW/dr(r, H_i) / r times (v_j - v_i) . d and (v_i - v_j) x d
                const float2 dw = kern_dw2<KERNEL>(make_float2(r * A.hinv, 1.f));
                const float g = other ? P2.z * A.f4 * dw.x * rinv : 0.f;
                const float wx = P1.x - A.vx, wy = P1.y - A.vy, wz = P1.z - A.vz;
                su += g * fmaf(wz, dz, fmaf(wy, dy, wx * dx));
                sx -= g * (wy * dz - wz * dy);
                sy -= g * (wz * dx - wx * dz);
                sz -= g * (wx * dy - wy * dx);
                continue;
            }
            const float hinv_j = P2.w; // 1 / H_j, correctly rounded once per particle (k_force_prep)
            const float hj2 = hinv_j * hinv_j;
            const float2 dw = kern_dw2<KERNEL>(__fmul2_rn(make_float2(r, r), make_float2(A.hinv, hinv_j)));
            const float Fi = A.f4 * dw.x;
            const float Fj = kern_sigma<KERNEL>() * hj2 * hj2 * dw.y;
            const float dvx = A.vx - P1.x, dvy = A.vy - P1.y, dvz = A.vz - P1.z;
            const float vr = fmaf(dvz, dz, fmaf(dvy, dy, dvx * dx)) * rinv;
            const float mu = fminf(vr, 0.f);
            const float vs = A.c + P1.w - 3.f * mu;
            const float Fbar = 0.5f * (Fi + Fj);
            if (MODE == MODE_CONDUCT) {
                // R21: m_j / (rho_i rho_j) * 4 k_i k_j / (k_i + k_j) * (T_i - T_j) * Fbar / r
                const float4 E = __ldg(a.ext + j); // kappa_j, T_j
                const float ks = A.al + E.x;
                const float kij = ks > 0.f ? 4.f * A.al * E.x * rcp_ftz(ks) : 0.f;
                const float e = other ? P2.z * rcp_ftz(A.rho * P2.x) * kij * (A.u - E.y) * Fbar * rinv : 0.f;
                su += e;
                continue;
            }
            float Pi, cond = 0.f;
            if (MODE == MODE_IMPROVED) {
                const float4 E = __ldg(a.ext + j);                         // alpha_j, f_j, u_j
                const float rbi = 2.f * rcp_ftz(A.rho + P2.x);                    // 1 / rho_bar
                Pi = -0.25f * (A.al + E.x) * vs * mu * rbi * 0.5f * (A.fb + E.y);               // R9 with R18, R19
                const float Pj = a.gm1 * P2.x * E.z;
                cond = a.alpha_cond * sqrt_ftz(fabsf(A.P - Pj) * rbi) * (A.u - E.z) * Fbar * rbi;   // R20
            } else {
                Pi = -alpha * vs * mu * rcp_ftz(A.rho + P2.x);
            }
            const float AiFi = A.A * Fi;
            const float pv = Pi * Fbar;
            // select, not multiply by zero: a lone particle has Omega = 0, hence A = inf
            const float tr = other ? P2.z * (AiFi + fmaf(P2.y, Fj, pv)) * rinv : 0.f;
            const float du = other ? P2.z * (fmaf(0.5f, pv, AiFi) * vr + cond) : 0.f;
            sx = fmaf(-tr, dx, sx);
            sy = fmaf(-tr, dy, sy);
            sz = fmaf(-tr, dz, sz);
            su += du;
            A.pvs = fmaxf(A.pvs, other ? vs : 0.f);
        }
    }
    A.px += (double)sx; A.py += (double)sy; A.pz += (double)sz; A.pdu += (double)su;
    A.cn += m;
    A.cnt = base;
}

template <int KERNEL, int MODE>
__device__ __forceinline__ void drain_any(const ForceArgs &a, uint32_t q0, ForceLane &A, int n, const Frame &fr)
{
    if (fr.pairwrap) drain<KERNEL, 2, MODE>(a, q0, A, n, fr);
    else if (fr.rec) drain<KERNEL, 1, MODE>(a, q0, A, n, fr);
    else drain<KERNEL, 0, MODE>(a, q0, A, n, fr);
}

// Test the candidate pairs of the gathered chunk against this lane's active (symmetric set, R10):
// hit if r^2 < max(H_i, H_j)^2; a hit pushes the candidate's sorted slot onto the lane's queue.
template <int KERNEL, bool PAIRWRAP, int MODE>
__device__ __forceinline__ void consume_chunk(const ForceArgs &a, const float4 *__restrict__ slotp,
                                              const uint32_t *__restrict__ gp, uint32_t q0, ForceLane &A,
                                              int s, int f, bool live, const Frame &fr)
{
    const int steps = (SPH_CH / 2) / f;
    const float4 *cp = slotp + s;
    uint32_t ga = smem_u32(gp + 2 * s);
    const float L = a.L;
    const float xf = PAIRWRAP ? A.xi : recentre(A.xi, fr.thx, L);
    const float yf = PAIRWRAP ? A.yi : recentre(A.yi, fr.thy, L);
    const float zf = PAIRWRAP ? A.zi : recentre(A.zi, fr.thz, L);
    const float2 nx = make_float2(-xf, -xf), ny = make_float2(-yf, -yf), nz = make_float2(-zf, -zf);
    for (int t0 = 0; t0 < steps; t0 += SPH_QSTEP_FORCE) {
        const int nt = min(SPH_QSTEP_FORCE, steps - t0);
        const int mx = __reduce_max_sync(FULLMASK, A.cnt);
        if (mx + 2 * nt > SPH_QCAP_FORCE) {
            const int mn = __reduce_min_sync(FULLMASK, live ? A.cnt : 0x7fffffff);
            drain_any<KERNEL, MODE>(a, q0, A, max(mn, mx + 2 * nt - SPH_QCAP_FORCE), fr);
        }
        uint32_t qw = q0 + (uint32_t)A.cnt * 128u;
#pragma unroll 2
        for (int t = 0; t < nt; t++) {
            const float4 c0 = cp[0], c1 = cp[SPH_CH / 2]; // (x0,x1,y0,y1) (z0,z1,H0^2,H1^2)
            cp += f;
            float2 r2;
            if (PAIRWRAP) {
                const float dx0 = image_diff(A.xi, c0.x, L), dx1 = image_diff(A.xi, c0.y, L);
                const float dy0 = image_diff(A.yi, c0.z, L), dy1 = image_diff(A.yi, c0.w, L);
                const float dz0 = image_diff(A.zi, c1.x, L), dz1 = image_diff(A.zi, c1.y, L);
                r2 = make_float2(fmaf(dz0, dz0, fmaf(dy0, dy0, dx0 * dx0)), fmaf(dz1, dz1, fmaf(dy1, dy1, dx1 * dx1)));
            } else {
                const float2 dx = __fadd2_rn(make_float2(c0.x, c0.y), nx), dy = __fadd2_rn(make_float2(c0.z, c0.w), ny);
                const float2 dz = __fadd2_rn(make_float2(c1.x, c1.y), nz);
                r2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
            }
            const float2 hj2 = make_float2(c1.z, c1.w); // H_j^2 (squared once per candidate by the gather)
            // symmetric set r < max(H_i, H_j) (R10); the velocity gradients gather over the own support only (R17)
            if (r2.x < (MODE == MODE_GRADV ? A.h2 : fmaxf(A.h2, hj2.x))) {
                sts_u32(qw, lds_u32(ga));
                qw += 128u;
            }
            if (r2.y < (MODE == MODE_GRADV ? A.h2 : fmaxf(A.h2, hj2.y))) {
                sts_u32(qw, lds_u32(ga + 4u));
                qw += 128u;
            }
            ga += 8u * (uint32_t)f;
        }
        A.cnt = (int)((qw - q0) >> 7);
    }
}

template <int KERNEL, int MODE>
__global__ void __launch_bounds__(SPH_THREADS, MODE == MODE_IMPROVED ? SPH_CTAS_FORCE - 1 : SPH_CTAS_FORCE) k_force(ForceArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ForceWarp &W = reinterpret_cast<ForceWarp *>(smem_raw)[warp];
    const float L = a.L;
    if (a.cnt->err | a.cnt->idx_err) return; // a precondition failed (ids, h, state, positions): compute nothing (uniform over the grid)
    const unsigned int n_groups = *a.n_groups;
    unsigned long long st_cands = 0, st_pairs = 0;
    const uint32_t q0 = smem_u32(W.q + lane); // shared-memory address of entry 0 of this lane's hit queue

    unsigned int gnext = 0, gend = 0; // this warp's block of consecutive groups
    for (;;) {
        if (gnext == gend) {
            if (lane == 0) gnext = atomicAdd(&a.cnt->work, (unsigned int)SPH_GBLOCK);
            gnext = __shfl_sync(FULLMASK, gnext, 0);
            if (gnext >= n_groups) break;
            gend = min(gnext + SPH_GBLOCK, n_groups);
        }
        const unsigned int grp = gnext++;
        const uint32_t i0 = a.gstart[grp];
        const uint32_t i1 = (grp + 1 < n_groups) ? a.gstart[grp + 1] : a.n_items;
        const int g = (int)(i1 - i0);
        const int f = streams_for(g);
        const bool live = lane < g * f;
        const int ai = live ? lane % g : 0, s = live ? lane / g : 0;
        ForceLane A;
        {
            const uint32_t slot = a.item_slot ? a.item_slot[i0 + ai] : i0 + ai;
            const float4 p0 = a.xyzh[slot], p1 = a.vc[2 * (size_t)slot], p2 = a.vc[2 * (size_t)slot + 1];
            A.slot = slot;
            A.xi = live ? p0.x : SPH_NANF; // dead lanes never hit
            A.yi = p0.y; A.zi = p0.z;
            A.h2 = p0.w * p0.w;
            A.hinv = 1.f / p0.w;
            const float h2i = A.hinv * A.hinv;
            A.f4 = kern_sigma<KERNEL>() * h2i * h2i;
            A.vx = p1.x; A.vy = p1.y; A.vz = p1.z; A.c = p1.w;
            A.rho = p2.x; A.A = p2.y;
            A.al = A.fb = A.u = A.P = 0.f;
            if (MODE == MODE_IMPROVED) {
                const float4 e = a.ext[slot];
                A.al = e.x; A.fb = e.y; A.u = e.z;
                A.P = a.gm1 * p2.x * e.z;
            }
            if (MODE == MODE_CONDUCT) {
                const float4 e = a.ext[slot];
                A.al = e.x; A.u = e.y; // kappa_i, T_i
            }
            A.px = A.py = A.pz = A.pdu = 0.0;
            A.pvs = 0.f;
            A.cn = A.cnt = 0;
            // bounding box and reach of the group
            const float inf = __int_as_float(0x7f800000);
            const float x0 = warp_min(live ? p0.x : inf), x1 = warp_max(live ? p0.x : -inf);
            const float y0 = warp_min(live ? p0.y : inf), y1 = warp_max(live ? p0.y : -inf);
            const float z0 = warp_min(live ? p0.z : inf), z1 = warp_max(live ? p0.z : -inf);
            const float hg = warp_max(live ? p0.w : 0.f);
            const float gcx = 0.5f * (x0 + x1), ghx = 0.5f * (x1 - x0) * (1.f + 1e-6f);
            const float gcy = 0.5f * (y0 + y1), ghy = 0.5f * (y1 - y0) * (1.f + 1e-6f);
            const float gcz = 0.5f * (z0 + z1), ghz = 0.5f * (z1 - z0) * (1.f + 1e-6f);

            WalkCtl ctl;
            ctl.sp = -1;
            unsigned long long cands = 0;
            Frame fr;
            fr.thx = fr.thy = fr.thz = __int_as_float(0x7f800000);
            fr.pairwrap = false;
            fr.rec = false;
            do {
                walk_batch<MODE != MODE_GRADV>(W.ws, ctl, a.nodes, a.node_hmax, L, gcx, gcy, gcz, ghx, ghy, ghz, hg);
                cands += ctl.total;
                // queued hits of an earlier batch are evaluated in the frame they were found in
                if (ctl.pairwrap != fr.pairwrap || ctl.thx != fr.thx || ctl.thy != fr.thy || ctl.thz != fr.thz) {
                    drain_any<KERNEL, MODE>(a, q0, A, __reduce_max_sync(FULLMASK, A.cnt), fr);
                    fr.thx = ctl.thx; fr.thy = ctl.thy; fr.thz = ctl.thz; fr.pairwrap = ctl.pairwrap;
                    fr.rec = ctl.thx < 1e30f || ctl.thy < 1e30f || ctl.thz < 1e30f;
                }
                const uint32_t nch = (ctl.total + SPH_CH - 1) / SPH_CH;
                GatherCtl gc;
                gc.kseg = 0;
                // (the register-staged gather pipeline of the density kernel measured slower here: 85.8 vs 76.3 ms)
                for (uint32_t c = 0; c < nch; c++) {
                    GatherRegs G;
                    gather_load(W.ws, ctl, gc, c, G, a.xyzh);
                    gather_store<true, true>(ctl, G, W.slot, W.gidx, L);
                    if (fr.pairwrap) consume_chunk<KERNEL, true, MODE>(a, W.slot, W.gidx, q0, A, s, f, live, fr);
                    else consume_chunk<KERNEL, false, MODE>(a, W.slot, W.gidx, q0, A, s, f, live, fr);
                }
            } while (ctl.sp > 0);
            drain_any<KERNEL, MODE>(a, q0, A, __reduce_max_sync(FULLMASK, A.cnt), fr);
            // cross-stream totals
            double X = A.px, Y = A.py, Z = A.pz, U = A.pdu;
            float V = A.pvs;
            int cn = A.cn;
            for (int d = 1; d < f; d <<= 1) {
                const bool take = live && s + d < f;
                const int from = take ? lane + g * d : lane;
                const double tX = __shfl_sync(FULLMASK, X, from), tY = __shfl_sync(FULLMASK, Y, from);
                const double tZ = __shfl_sync(FULLMASK, Z, from), tU = __shfl_sync(FULLMASK, U, from);
                const float tV = __shfl_sync(FULLMASK, V, from);
                const int tn = __shfl_sync(FULLMASK, cn, from);
                if (take) { X += tX; Y += tY; Z += tZ; U += tU; V = fmaxf(V, tV); cn += tn; }
            }
            // a11: scatter to the caller's particle id
            if (lane < g) {
                const uint32_t id = a.perm[slot];
                if (MODE == MODE_GRADV) {
                    const double ir = 1.0 / (double)A.rho;
                    a.divv[id] = (float)(U * ir);
                    a.curlv[3 * (size_t)id] = (float)(X * ir);
                    a.curlv[3 * (size_t)id + 1] = (float)(Y * ir);
                    a.curlv[3 * (size_t)id + 2] = (float)(Z * ir);
                } else if (MODE == MODE_CONDUCT) {
                    a.dudt[id] = (float)U;
                } else {
                    a.acc[3 * (size_t)id] = (float)X;
                    a.acc[3 * (size_t)id + 1] = (float)Y;
                    a.acc[3 * (size_t)id + 2] = (float)Z;
                    a.dudt[id] = (float)U;
                    a.vsig[id] = V;
                }
                if (MODE == MODE_IMPROVED) { // R19: d alpha/dt = -(alpha - alpha_min) 2 l c / H + max(0, -div v)(alpha_max - alpha)
                    const float dv = a.divv[id];
                    a.dalpha[id] = -(A.al - a.alpha_min) * 2.f * a.decay_l * A.c * A.hinv + fmaxf(-dv, 0.f) * (a.alpha_max - A.al);
                }
            }
            unsigned long long pr = (lane < g) ? (unsigned long long)(cn - 1) : 0ull; // minus self
#pragma unroll
            for (int o = 16; o; o >>= 1) pr += __shfl_xor_sync(FULLMASK, pr, o);
            st_pairs += pr;
            st_cands += cands * (unsigned long long)g;
        }
    }
    if (lane == 0) {
        if (st_cands) atomicAdd(&a.cnt->force_cands, st_cands);
        if (st_pairs) atomicAdd(&a.cnt->force_pairs, st_pairs);
    }
}

// gather the caller-order state into the sorted float4 arrays the gather streams through shared memory
__global__ void k_force_prep(int64_t n, const uint32_t *__restrict__ perm, const float4 *__restrict__ xyzm,
                             const float *__restrict__ vel, const float *__restrict__ u, const float *__restrict__ h,
                             const float *__restrict__ rho, const float *__restrict__ omega, float gamma, float half_box,
                             float4 *__restrict__ xyzh, float4 *__restrict__ vc, SphCounters *cnt,
                             const float *__restrict__ alpha, const float *__restrict__ divv, const float *__restrict__ curlv,
                             int balsara, float4 *__restrict__ ext, float kappa0, float kappa_exp, int conduct,
                             const SphNode *__restrict__ nodes, const uint32_t *__restrict__ slot_leaf, float *__restrict__ hmax)
{
    // u, omega may be NULL (velocity-gradient pass: only positions, h, velocities, rho and masses are used);
    // alpha != NULL: improved-SPH state record (alpha, shear limiter f of R18, u) per particle
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    // largest support radius inside every octree node (hmax != NULL; zeroed before): the lanes that share a leaf send
    // one value up the parent chain with integer atomicMax (H > 0: the float bit patterns order like integers)
    if (hmax) {
        const uint32_t leaf = i < n ? slot_leaf[i] : 0xffffffffu;
        const float H = i < n ? h[perm[i]] : 0.f;
        const unsigned grp = __match_any_sync(0xffffffffu, leaf);
        const int mb = __reduce_max_sync(grp, H > 0.f ? __float_as_int(H) : 0);
        if (i < n && (threadIdx.x & 31) == __ffs(grp) - 1 && mb > 0) {
            uint32_t cur = leaf;
            for (;;) {
                if (__float_as_int(__ldcg(hmax + cur)) >= mb) break;
                const int old = atomicMax(reinterpret_cast<int *>(hmax) + cur, mb);
                if (cur == 0 || old >= mb) break;
                cur = nodes[cur].parent;
            }
        }
    }
    if (i >= n) return;
    uint32_t id = perm[i];
    float4 p = xyzm[i];
    float ui = u ? u[id] : 0.f, ri = rho[id];
    // preconditions on the state of ALL particles (inactive neighbours contribute, R12): 0 < H < box / 2, rho > 0,
    // u >= 0, everything finite (a comparison with NaN is false)
    {
        const float inf = __int_as_float(0x7f800000);
        const float H = h[id], om = omega ? omega[id] : 1.f;
        const float v2 = vel ? fabsf(vel[3 * (int64_t)id]) + fabsf(vel[3 * (int64_t)id + 1]) + fabsf(vel[3 * (int64_t)id + 2]) : 0.f;
        if (!(H > 0.f) || !(H < inf)) atomicOr(&cnt->err, SPH_ERR_H);
        else if (!(H < half_box)) atomicOr(&cnt->err, SPH_ERR_HRANGE);
        if (!(ri > 0.f) || !(ri < inf) || !(ui >= 0.f) || !(ui < inf) || !(fabsf(om) < inf) || !(v2 < inf)) atomicOr(&cnt->err, SPH_ERR_STATE);
    }
    float c = sqrtf(gamma * (gamma - 1.f) * ui);
    float A = omega ? (gamma - 1.f) * ui / (omega[id] * ri) : 0.f; // P/(Omega rho^2), P = (gamma-1) rho u
    xyzh[i] = make_float4(p.x, p.y, p.z, h[id]);
    vc[2 * i] = vel ? make_float4(vel[3 * (int64_t)id], vel[3 * (int64_t)id + 1], vel[3 * (int64_t)id + 2], c) : make_float4(0.f, 0.f, 0.f, c);
    if (conduct) ext[i] = make_float4(kappa0 * powf(ui, kappa_exp), ui, 0.f, 0.f); // R21: kappa = kappa_0 T^e, T = u
    vc[2 * i + 1] = make_float4(ri, A, p.w, 1.f / h[id]);
    if (alpha) {
        const float inf = __int_as_float(0x7f800000);
        const float al = alpha[id], dv = divv[id];
        const float cx = curlv[3 * (int64_t)id], cy = curlv[3 * (int64_t)id + 1], cz = curlv[3 * (int64_t)id + 2];
        const float cm = sqrtf(fmaf(cz, cz, fmaf(cy, cy, cx * cx)));
        if (!(al >= 0.f) || !(al < inf) || !(fabsf(dv) < inf) || !(cm < inf)) atomicOr(&cnt->err, SPH_ERR_STATE);
        const float fb = balsara ? fabsf(dv) / (fabsf(dv) + cm + 1e-4f * c / h[id]) : 1.f; // R18
        ext[i] = make_float4(al, fb, ui, 0.f);
    }
}

__global__ void k_zero_hmax(const SphCounters *cnt, float *__restrict__ hmax)
{
    uint32_t nn = cnt->n_nodes;
    for (uint32_t nd = blockIdx.x * blockDim.x + threadIdx.x; nd < nn; nd += gridDim.x * blockDim.x) hmax[nd] = 0.f;
}

template <int KERNEL, int MODE>
int launch(sph_ctx *ctx, const ForceArgs &a, int64_t est_groups)
{
    size_t dyn = sizeof(ForceWarp) * SPH_WARPS;
    auto kfn = k_force<KERNEL, MODE>;
    SPH_CUDA(ctx, cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
    int per_sm = 1;
    SPH_CUDA(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kfn, SPH_THREADS, dyn));
    if (per_sm < 1) return sph_fail(ctx, SPH_E_INTERNAL, "k_force does not fit on an SM");
    int64_t grid = (int64_t)ctx->device_sms * per_sm;
    int64_t need = (est_groups + SPH_WARPS * SPH_GBLOCK - 1) / (SPH_WARPS * SPH_GBLOCK);
    if (need < grid) grid = need > 0 ? need : 1;
    kfn<<<(int)grid, SPH_THREADS, dyn, ctx->stream>>>(a);
    SPH_CUDA(ctx, cudaGetLastError());
    return SPH_OK;
}

} // namespace

// mode: MODE_BASE (sph_hydro_force), MODE_IMPROVED (sph_hydro_force_improved), MODE_GRADV (sph_velocity_gradients)
int sph_force_launch(sph_ctx *ctx, int mode, bool subset, int64_t n_items, const float *vel, const float *u, const float *h,
                     const float *rho, const float *omega, float *acc, float *dudt, float *vsig, const float *alpha,
                     const float *divv, const float *curlv, const sph_improved_params *ip, float *dalpha, float *divv_out,
                     float *curlv_out, float kappa0, float kappa_exp)
{
    cudaStream_t st = ctx->stream;
    const int64_t n = ctx->n;
    const int T = 256;
    if ((mode == MODE_IMPROVED || mode == MODE_CONDUCT) && !ctx->f_ext) {
        SPH_CUDA(ctx, cudaMalloc((void **)&ctx->f_ext, sizeof(float4) * (size_t)ctx->cap_n));
    }
    cudaEventRecord(ctx->ev[4], st);
    const bool need_hmax = mode != MODE_GRADV; // the symmetric pair set needs the largest support radius inside every node
    if (need_hmax) {
        k_zero_hmax<<<ctx->device_sms * 4, 256, 0, st>>>(ctx->cnt, ctx->node_hmax);
        ctx->launches++;
    }
    k_force_prep<<<(int)((n + T - 1) / T), T, 0, st>>>(n, ctx->perm, ctx->xyzm, vel, u, h, rho, omega, ctx->prm.gamma,
                                                       0.5f * ctx->prm.box, ctx->f_xyzh, ctx->f_vc, ctx->cnt,
                                                       mode == MODE_IMPROVED ? alpha : nullptr, divv, curlv,
                                                       ip ? ip->balsara : 0, ctx->f_ext, kappa0, kappa_exp, mode == MODE_CONDUCT,
                                                       ctx->nodes, ctx->slot_leaf, need_hmax ? ctx->node_hmax : nullptr);
    ctx->launches++;
    sph_reset_counters(ctx, 1, subset);
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
    a.ext = ctx->f_ext;
    a.gm1 = ctx->prm.gamma - 1.f;
    a.alpha_cond = ip ? ip->alpha_cond : 0.f;
    a.alpha_min = ip ? ip->alpha_min : 0.f;
    a.alpha_max = ip ? ip->alpha_max : 0.f;
    a.decay_l = ip ? ip->decay_l : 0.f;
    a.dalpha = dalpha;
    a.divv = mode == MODE_GRADV ? divv_out : const_cast<float *>(divv);
    a.curlv = curlv_out;
    int64_t est_groups = n_items; // (an upper bound: the group count stays on the device)
    cudaEventRecord(ctx->ev[6], st);
    int rc;
    const bool cubic = ctx->prm.kernel == SPH_KERNEL_CUBIC;
    if (mode == MODE_BASE) rc = cubic ? launch<SPH_KERNEL_CUBIC, MODE_BASE>(ctx, a, est_groups) : launch<SPH_KERNEL_WC6, MODE_BASE>(ctx, a, est_groups);
    else if (mode == MODE_IMPROVED) rc = cubic ? launch<SPH_KERNEL_CUBIC, MODE_IMPROVED>(ctx, a, est_groups) : launch<SPH_KERNEL_WC6, MODE_IMPROVED>(ctx, a, est_groups);
    else if (mode == MODE_GRADV) rc = cubic ? launch<SPH_KERNEL_CUBIC, MODE_GRADV>(ctx, a, est_groups) : launch<SPH_KERNEL_WC6, MODE_GRADV>(ctx, a, est_groups);
    else rc = cubic ? launch<SPH_KERNEL_CUBIC, MODE_CONDUCT>(ctx, a, est_groups) : launch<SPH_KERNEL_WC6, MODE_CONDUCT>(ctx, a, est_groups);
    cudaEventRecord(ctx->ev[7], st);
    ctx->ev_set[3] = true;
    ctx->launches++;
    return rc;
}
