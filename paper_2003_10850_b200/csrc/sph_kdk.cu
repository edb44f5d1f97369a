// sph_kdk.cu -- SURVEY.md §8(f)-3: kick-drift-kick time integration with power-of-two time bins, the driver that
// produces the active lists of the hot path step after step.
//
// "Gadget3 ... uses an adaptive time-stepping scheme: particles are assigned to time bins of power-of-two length"
// and only the particles whose bin is due ("active particles") are updated (PAPER.md:37 §1, :84-86 §2.2: "the
// number of active particles ... can be as small as one"; :114 §3).  The paper gives no formulas: reading R22 of
// DESIGN.md, the kick-drift-kick scheme of the Gadget lineage [2] restated from its published description.
//
// Timeline: T = 2^(n_bins-1) ticks per dt_max; a particle of bin b steps s_b = T >> b ticks.  One call of
// sph_kdk_step advances to the next tick at which a step ends (the smallest occupied step), drifts ALL particles
// there, runs the hot path (index build, density with the last h as the guess, hydro force with drifted
// velocities and energies) for the particles whose step ends, closes their step (second half kick), gives them a
// new bin from the time-step criterion and opens the next step (first half kick).
#include <math.h>

#include "sph_internal.cuh"

namespace {

struct KdkConst {
    float box, delta;   // periodic box edge; length of one tick
    int T, n_bins;      // ticks per dt_max; number of bins
    float dt_max, courant, eta;
};

// dt = min(C H / vsig, sqrt(2 eta H / |a|)) -> smallest b with dt_max / 2^b <= dt, clamped to [0, n_bins - 1] (R22)
__device__ __forceinline__ int bin_of(const KdkConst &k, float H, float vsig, float ax, float ay, float az)
{
    const float a = sqrtf(fmaf(az, az, fmaf(ay, ay, ax * ax)));
    float dt = vsig > 0.f ? k.courant * H / vsig : __int_as_float(0x7f800000);
    if (a > 0.f) dt = fminf(dt, sqrtf(2.f * k.eta * H / a));
    const float x = log2f(k.dt_max / dt); // -inf for dt = inf
    int b = x > 0.f ? (int)ceilf(x) : 0;
    return min(max(b, 0), k.n_bins - 1);
}

// all particles at tick 0 (after the first force pass): bin, step begin, first half kick
__global__ void k_kdk_open_all(int64_t n, KdkConst k, const float *__restrict__ h, const float *__restrict__ vsig,
                               const float *__restrict__ acc, const float *__restrict__ dudt, float *__restrict__ vel,
                               float *__restrict__ u, int32_t *__restrict__ bin, int32_t *__restrict__ tbegin, unsigned int *bmax)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float ax = acc[3 * i], ay = acc[3 * i + 1], az = acc[3 * i + 2];
    const int b = bin_of(k, h[i], vsig[i], ax, ay, az);
    const float hk = 0.5f * (float)(k.T >> b) * k.delta;
    vel[3 * i] = fmaf(ax, hk, vel[3 * i]);
    vel[3 * i + 1] = fmaf(ay, hk, vel[3 * i + 1]);
    vel[3 * i + 2] = fmaf(az, hk, vel[3 * i + 2]);
    u[i] = fmaf(dudt[i], hk, u[i]);
    bin[i] = b;
    tbegin[i] = 0;
    atomicMax(bmax, (unsigned int)b);
}

// drift all particles by ds ticks to t1; drifted velocity and energy for the force pass; flag the particles whose step ends
__global__ void k_kdk_drift(int64_t n, KdkConst k, int ds, int t1, float *__restrict__ pos, const float *__restrict__ vel,
                            const float *__restrict__ u, const float *__restrict__ acc, const float *__restrict__ dudt,
                            const int32_t *__restrict__ bin, const int32_t *__restrict__ tbegin, float *__restrict__ vpred,
                            float *__restrict__ upred, uint32_t *__restrict__ flag)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float dt = (float)ds * k.delta;
    const int s = k.T >> bin[i];
    const float since_mid = ((float)(t1 - tbegin[i]) - 0.5f * (float)s) * k.delta; // time since the middle of the step
#pragma unroll
    for (int c = 0; c < 3; c++) {
        const float v = vel[3 * i + c];
        float x = fmaf(v, dt, pos[3 * i + c]);
        if (x >= k.box) x -= k.box;
        if (x < 0.f) x += k.box;
        if (!(x < k.box)) x = 0.f; // (-tiny + box rounds to box)
        pos[3 * i + c] = x;
        vpred[3 * i + c] = fmaf(acc[3 * i + c], since_mid, v);
    }
    upred[i] = fmaxf(fmaf(dudt[i], since_mid, u[i]), 0.f);
    flag[i] = (t1 - tbegin[i] == s) ? 1u : 0u;
}

// close the step of the active particles (second half kick), choose the new bin, open the next step (first half kick)
__global__ void k_kdk_close_open(int64_t na, KdkConst k, int t1, const int32_t *__restrict__ active, const float *__restrict__ h,
                                 const float *__restrict__ vsig, const float *__restrict__ acc, const float *__restrict__ dudt,
                                 float *__restrict__ vel, float *__restrict__ u, int32_t *__restrict__ bin,
                                 int32_t *__restrict__ tbegin)
{
    const int64_t kk = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (kk >= na) return;
    const int64_t i = active[kk];
    const float ax = acc[3 * i], ay = acc[3 * i + 1], az = acc[3 * i + 2];
    const int b0 = bin[i];
    int b = bin_of(k, h[i], vsig[i], ax, ay, az);
    // a longer step only one bin at a time, and only where the timeline is aligned with it
    if (b < b0) b = (t1 % (k.T >> (b0 - 1)) == 0) ? b0 - 1 : b0;
    const float hk = 0.5f * (float)((k.T >> b0) + (k.T >> b)) * k.delta; // second half of the old step + first half of the new one
    vel[3 * i] = fmaf(ax, hk, vel[3 * i]);
    vel[3 * i + 1] = fmaf(ay, hk, vel[3 * i + 1]);
    vel[3 * i + 2] = fmaf(az, hk, vel[3 * i + 2]);
    u[i] = fmaxf(fmaf(dudt[i], hk, u[i]), 0.f);
    bin[i] = b;
    tbegin[i] = t1;
}

// acc += gravity for the listed particles (active == NULL: all)
__global__ void k_kdk_add_gravity(int64_t na, const int32_t *__restrict__ active, const float *__restrict__ grav, float *__restrict__ acc)
{
    const int64_t kk = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (kk >= na) return;
    const int64_t i = active ? active[kk] : kk;
    acc[3 * i] += grav[3 * i];
    acc[3 * i + 1] += grav[3 * i + 1];
    acc[3 * i + 2] += grav[3 * i + 2];
}

__global__ void k_kdk_bmax(int64_t n, const int32_t *__restrict__ bin, unsigned int *bmax)
{
    unsigned int m = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) m = max(m, (unsigned int)bin[i]);
    m = __reduce_max_sync(0xffffffffu, m);
    if ((threadIdx.x & 31) == 0) atomicMax(bmax, m);
}

__global__ void k_iota(int64_t n, int32_t *a)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = (int32_t)i;
}

int check(sph_ctx *ctx, int64_t n, const sph_kdk_params *p, const sph_kdk_state *s, KdkConst &k)
{
    if (!p || !s || n < 0) return sph_fail(ctx, SPH_E_ARG, "sph_kdk: NULL params/state or n < 0");
    if (!(p->dt_max > 0.f) || p->n_bins < 1 || p->n_bins > 24 || !(p->courant > 0.f) || !(p->eta > 0.f) || !(p->n_ngb_target > 0.f) ||
        !(p->n_ngb_tol >= 0.f))
        return sph_fail(ctx, SPH_E_ARG, "sph_kdk: bad sph_kdk_params");
    if (p->grav_G < 0.f || (p->grav_G > 0.f && (!(p->grav_rs > 0.f) || !(p->grav_rcut > 0.f) || !(p->grav_eps >= 0.f) || !(p->grav_theta >= 0.f))))
        return sph_fail(ctx, SPH_E_ARG, "sph_kdk: bad gravity parameters in sph_kdk_params");
    if (n > 0 && (!s->pos || !s->vel || !s->u || !s->h || !s->rho || !s->omega || !s->ngb || !s->acc || !s->dudt || !s->vsig ||
                  !s->vpred || !s->upred || !s->bin || !s->tbegin || !s->active))
        return sph_fail(ctx, SPH_E_ARG, "sph_kdk: NULL array in sph_kdk_state");
    k.box = ctx->prm.box;
    k.T = 1 << (p->n_bins - 1);
    k.n_bins = p->n_bins;
    k.delta = p->dt_max / (float)k.T;
    k.dt_max = p->dt_max;
    k.courant = p->courant;
    k.eta = p->eta;
    return SPH_OK;
}

// short-range gravity of the listed particles added to their hydro acceleration (grav_G > 0); the active groups of the
// density pass are still valid (act_keep set by the caller)
int add_gravity(sph_ctx *ctx, int64_t n, const sph_kdk_params *p, const sph_kdk_state *s, const int32_t *active, int64_t na)
{
    if (!(p->grav_G > 0.f)) return SPH_OK;
    int rc;
    if (ctx->kdk_grav_cap < n) {
        ctx->kdk_grav_cap = 0;
        if (ctx->kdk_grav) cudaFree(ctx->kdk_grav);
        ctx->kdk_grav = nullptr;
        SPH_CUDA(ctx, cudaMalloc((void **)&ctx->kdk_grav, sizeof(float) * 3 * (size_t)n));
        ctx->kdk_grav_cap = n;
    }
    if ((rc = sph_gravity_short(ctx, active, active ? na : -1, p->grav_G, p->grav_rs, p->grav_rcut, p->grav_eps, p->grav_theta, ctx->kdk_grav)))
        return rc;
    const int64_t cnt = active ? na : n;
    if (cnt > 0) k_kdk_add_gravity<<<(int)((cnt + 255) / 256), 256, 0, ctx->stream>>>(cnt, active, ctx->kdk_grav, s->acc);
    ctx->launches++;
    return SPH_OK;
}

} // namespace

extern "C" {

int sph_kdk_init(sph_ctx *ctx, int64_t n, float mass_scalar, const sph_kdk_params *p, const sph_kdk_state *s)
{
    if (!ctx) return SPH_E_ARG;
    KdkConst k;
    int rc = check(ctx, n, p, s, k);
    if (rc) return rc;
    ctx->kdk_tick = 0;
    ctx->kdk_refreshed = 0;
    if (n == 0) return SPH_OK;
    cudaStream_t st = ctx->stream;
    const int T = 256, G = (int)((n + T - 1) / T);
    if ((rc = sph_build_index(ctx, n, s->pos, nullptr, mass_scalar))) return rc;
    if ((rc = sph_active_reserve(ctx, n))) return rc; // active lists of any length without reallocation later
    int64_t unconv = 0;
    rc = sph_density(ctx, nullptr, -1, p->n_ngb_target, p->n_ngb_tol, s->h, s->rho, s->omega, s->ngb, nullptr, &unconv);
    if (rc != SPH_OK && rc != SPH_W_NOCONV) return rc;
    const int rcd = rc;
    if ((rc = sph_hydro_force(ctx, nullptr, -1, s->vel, s->u, s->h, s->rho, s->omega, s->acc, s->dudt, s->vsig))) return rc;
    if ((rc = add_gravity(ctx, n, p, s, nullptr, n))) return rc;
    SPH_CUDA(ctx, cudaMemsetAsync(&ctx->cnt->work, 0, sizeof(unsigned int), st)); // (reused as the bin maximum between calls of the gather kernels)
    k_kdk_open_all<<<G, T, 0, st>>>(n, k, s->h, s->vsig, s->acc, s->dudt, s->vel, s->u, s->bin, s->tbegin, &ctx->cnt->work);
    ctx->launches++;
    SPH_CUDA(ctx, cudaGetLastError());
    return rcd;
}

int sph_kdk_step(sph_ctx *ctx, int64_t n, float mass_scalar, const sph_kdk_params *p, const sph_kdk_state *s,
                 int64_t *tick_host, int64_t *n_active_host)
{
    if (!ctx) return SPH_E_ARG;
    KdkConst k;
    int rc = check(ctx, n, p, s, k);
    if (rc) return rc;
    if (n_active_host) *n_active_host = 0;
    if (tick_host) *tick_host = ctx->kdk_tick;
    if (n == 0) return SPH_OK;
    cudaStream_t st = ctx->stream;
    const int T = 256, G = (int)((n + T - 1) / T);
    // the next tick at which a step ends: the smallest occupied step (host round trip 1 of 2 of a step)
    unsigned int hb[1] = {0};
    SPH_CUDA(ctx, cudaMemsetAsync(&ctx->cnt->work, 0, sizeof(unsigned int), st));
    k_kdk_bmax<<<ctx->device_sms * 4, T, 0, st>>>(n, s->bin, &ctx->cnt->work);
    SPH_CUDA(ctx, cudaMemcpyAsync(hb, &ctx->cnt->work, sizeof(unsigned int), cudaMemcpyDeviceToHost, st));
    SPH_CUDA(ctx, cudaStreamSynchronize(st));
    const int ds = k.T >> (int)hb[0];
    const int t1 = (int)ctx->kdk_tick + ds;
    // drift everybody, flag and list the particles whose step ends at t1 (ids ascending)
    if (n > ctx->cap_n) return sph_fail(ctx, SPH_E_NOINDEX, "sph_kdk_step before sph_kdk_init");
    k_kdk_drift<<<G, T, 0, st>>>(n, k, ds, t1, s->pos, s->vel, s->u, s->acc, s->dudt, s->bin, s->tbegin, s->vpred, s->upred, ctx->grp_mark);
    if ((rc = sph_scan_marks(ctx, ctx->grp_mark, n, nullptr, reinterpret_cast<uint32_t *>(s->active), &ctx->cnt->n_agroups))) return rc;
    unsigned int na = 0;
    SPH_CUDA(ctx, cudaMemcpyAsync(&na, &ctx->cnt->n_agroups, sizeof(unsigned int), cudaMemcpyDeviceToHost, st));
    SPH_CUDA(ctx, cudaStreamSynchronize(st));
    ctx->launches += 2;
    // the hot path for the active particles at their new positions
    // (few active particles: keep the tree and refresh it; the rebuild would be most of the step)
    const bool refresh = ctx->have_index && ctx->n == n && ctx->kdk_refreshed < p->refresh_max && (double)na < (double)p->rebuild_fraction * (double)n;
    if (refresh) {
        if ((rc = sph_refresh_index(ctx, n, s->pos))) return rc;
        ctx->kdk_refreshed++;
    } else {
        if ((rc = sph_build_index(ctx, n, s->pos, nullptr, mass_scalar))) return rc;
        ctx->kdk_refreshed = 0;
    }
    int64_t unconv = 0;
    const bool all = (int64_t)na == n;
    rc = sph_density(ctx, all ? nullptr : s->active, all ? -1 : (int64_t)na, p->n_ngb_target, p->n_ngb_tol, s->h, s->rho, s->omega, s->ngb,
                     nullptr, &unconv);
    if (rc != SPH_OK && rc != SPH_W_NOCONV) return rc;
    const int rcd = rc;
    ctx->act_keep = true; // the same active list: its groups are those of the density pass
    rc = sph_hydro_force(ctx, all ? nullptr : s->active, all ? -1 : (int64_t)na, s->vpred, s->upred, s->h, s->rho, s->omega, s->acc, s->dudt,
                         s->vsig);
    if (!rc) rc = add_gravity(ctx, n, p, s, all ? nullptr : s->active, (int64_t)na);
    ctx->act_keep = false;
    if (rc) return rc;
    if (all) k_iota<<<G, T, 0, st>>>(n, s->active);
    if (na) k_kdk_close_open<<<(int)((na + T - 1) / T), T, 0, st>>>((int64_t)na, k, t1, s->active, s->h, s->vsig, s->acc, s->dudt, s->vel, s->u,
                                                                   s->bin, s->tbegin);
    ctx->launches += 2;
    SPH_CUDA(ctx, cudaGetLastError());
    ctx->kdk_tick = t1;
    if (tick_host) *tick_host = t1;
    if (n_active_host) *n_active_host = (int64_t)na;
    return rcd;
}

} // extern "C"
