/* A plain C caller of libsph.so through include/sph.h alone (no Python, no ctypes mirror):
 * create -> build_index -> density -> hydro_force -> get_stats on a small jittered lattice, then the
 * error paths a C user meets.  Device memory through the CUDA runtime C API.  Prints "abi_smoke ok".
 * Built and run by tests/test_gpu_abi_c.py. */
#include <cuda_runtime_api.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include "sph.h"

#define CHECK(c)                                                        \
    do {                                                                \
        if (!(c)) {                                                     \
            fprintf(stderr, "abi_smoke: %s failed (line %d)\n", #c, __LINE__); \
            return 1;                                                   \
        }                                                               \
    } while (0)

static unsigned int lcg(unsigned int *s) { return *s = *s * 1664525u + 1013904223u; }
static float urand(unsigned int *s) { return (float)(lcg(s) >> 8) / 16777216.0f; }

static void *dev(const void *host, size_t bytes)
{
    void *p = NULL;
    if (cudaMalloc(&p, bytes) != cudaSuccess) return NULL;
    if (host && cudaMemcpy(p, host, bytes, cudaMemcpyHostToDevice) != cudaSuccess) return NULL;
    if (!host) cudaMemset(p, 0, bytes);
    return p;
}

int main(void)
{
    enum { S = 10, N = S * S * S };
    static float pos[N * 3], vel[N * 3], u[N], h[N], rho[N], om[N], acc[N * 3], du[N], vs[N];
    static int32_t ngb[N], st[N];
    unsigned int seed = 200310850u;
    const float d = 1.0f / S;
    for (int i = 0; i < N; i++) {
        int ix = i % S, iy = (i / S) % S, iz = i / (S * S);
        pos[3 * i] = (ix + 0.5f + 0.5f * (urand(&seed) - 0.5f)) * d;
        pos[3 * i + 1] = (iy + 0.5f + 0.5f * (urand(&seed) - 0.5f)) * d;
        pos[3 * i + 2] = (iz + 0.5f + 0.5f * (urand(&seed) - 0.5f)) * d;
        for (int a = 0; a < 3; a++) vel[3 * i + a] = 0.1f * (urand(&seed) - 0.5f);
        u[i] = 1.0f + urand(&seed);
        h[i] = 0.2481f; /* (3 * 64 / (4 pi N))^(1/3) */
    }
    sph_params p = {SPH_KERNEL_CUBIC, 1.0f, 5.0f / 3.0f, 1.0f, 0, 64, 0, 0};
    sph_ctx *ctx = NULL;
    CHECK(sph_create(&ctx, &p, NULL) == SPH_OK && ctx);
    float *d_pos = dev(pos, sizeof pos), *d_vel = dev(vel, sizeof vel), *d_u = dev(u, sizeof u), *d_h = dev(h, sizeof h);
    float *d_rho = dev(NULL, sizeof rho), *d_om = dev(NULL, sizeof om), *d_acc = dev(NULL, sizeof acc);
    float *d_du = dev(NULL, sizeof du), *d_vs = dev(NULL, sizeof vs);
    int32_t *d_ngb = dev(NULL, sizeof ngb), *d_st = dev(NULL, sizeof st);
    CHECK(d_pos && d_vel && d_u && d_h && d_rho && d_om && d_acc && d_du && d_vs && d_ngb && d_st);

    /* before the index exists */
    int64_t unconv = -1;
    CHECK(sph_density(ctx, NULL, -1, 64.f, 2.f, d_h, d_rho, d_om, d_ngb, d_st, &unconv) == SPH_E_NOINDEX);
    CHECK(sph_last_error(ctx)[0] != 0);

    CHECK(sph_build_index(ctx, N, d_pos, NULL, 1.0f / N) == SPH_OK);
    CHECK(sph_density(ctx, NULL, -1, 64.f, 2.f, d_h, d_rho, d_om, d_ngb, d_st, &unconv) == SPH_OK && unconv == 0);
    CHECK(sph_hydro_force(ctx, NULL, -1, d_vel, d_u, d_h, d_rho, d_om, d_acc, d_du, d_vs) == SPH_OK);
    sph_stats s;
    CHECK(sph_get_stats(ctx, &s) == SPH_OK);
    CHECK(s.n == N && s.n_nodes > 8 && s.n_groups > 0 && s.launches > 0 && s.node_pool_overflow == 0);
    CHECK(s.dens_evals >= N && s.dens_pairs > 40 * (int64_t)N && s.force_pairs > 40 * (int64_t)N);
    CHECK(s.t_density_kernel_ms > 0.f && s.t_force_kernel_ms > 0.f && s.t_index_ms > 0.f);
    CHECK(cudaMemcpy(rho, d_rho, sizeof rho, cudaMemcpyDeviceToHost) == cudaSuccess);
    CHECK(cudaMemcpy(ngb, d_ngb, sizeof ngb, cudaMemcpyDeviceToHost) == cudaSuccess);
    CHECK(cudaMemcpy(st, d_st, sizeof st, cudaMemcpyDeviceToHost) == cudaSuccess);
    CHECK(cudaMemcpy(acc, d_acc, sizeof acc, cudaMemcpyDeviceToHost) == cudaSuccess);
    double mean = 0.0, px = 0.0, pa = 0.0;
    for (int i = 0; i < N; i++) {
        CHECK(rho[i] > 0.5f && rho[i] < 2.0f && ngb[i] > 30 && ngb[i] < 120 && (st[i] & SPH_ST_CONVERGED));
        mean += rho[i] / N;
        px += acc[3 * i];
        pa += fabs(acc[3 * i]);
    }
    CHECK(fabs(mean - 1.0) < 0.05);  /* density = m n within the lattice bound */
    CHECK(fabs(px) < 1e-4 * pa);     /* momentum: all active, pair terms antisymmetric */

    /* the same positions through sph_refresh_index: the same tree, hence the same integers */
    static int32_t ngb2[N];
    CHECK(sph_refresh_index(ctx, N - 1, d_pos) == SPH_E_ARG);
    CHECK(sph_refresh_index(ctx, N, d_pos) == SPH_OK);
    CHECK(cudaMemcpy(d_h, h, sizeof h, cudaMemcpyHostToDevice) == cudaSuccess);
    CHECK(sph_density(ctx, NULL, -1, 64.f, 2.f, d_h, d_rho, d_om, d_ngb, d_st, &unconv) == SPH_OK && unconv == 0);
    CHECK(cudaMemcpy(ngb2, d_ngb, sizeof ngb2, cudaMemcpyDeviceToHost) == cudaSuccess);
    for (int i = 0; i < N; i++) CHECK(ngb2[i] == ngb[i]);

    /* flags -> ascending id list, with the context's scratch and with the fixed device scratch */
    {
        static uint32_t fl[N];
        static int32_t idl[2][N];
        uint32_t cnt[2] = {77u, 77u};
        int want = 0;
        for (int i = 0; i < N; i++) { fl[i] = (i % 3 == 1) || (i > N - 5); want += (int)fl[i]; }
        uint32_t *d_fl = dev(fl, sizeof fl), *d_cnt = dev(NULL, sizeof cnt);
        int32_t *d_id0 = dev(NULL, sizeof idl[0]), *d_id1 = dev(NULL, sizeof idl[1]);
        CHECK(d_fl && d_cnt && d_id0 && d_id1);
        CHECK(sph_compact_flags(ctx, N, d_fl, d_id0, d_cnt) == SPH_OK);
        CHECK(sph_compact_flags_noalloc(ctx, N, d_fl, d_id1, d_cnt + 1) == SPH_OK);
        CHECK(sph_compact_flags_noalloc(ctx, (int64_t)SPH_COMPACT_NOALLOC_MAX + 1, d_fl, d_id1, d_cnt + 1) == SPH_E_ARG);
        CHECK(cudaDeviceSynchronize() == cudaSuccess);
        CHECK(cudaMemcpy(cnt, d_cnt, sizeof cnt, cudaMemcpyDeviceToHost) == cudaSuccess);
        CHECK(cudaMemcpy(idl[0], d_id0, sizeof idl[0], cudaMemcpyDeviceToHost) == cudaSuccess);
        CHECK(cudaMemcpy(idl[1], d_id1, sizeof idl[1], cudaMemcpyDeviceToHost) == cudaSuccess);
        CHECK((int)cnt[0] == want && (int)cnt[1] == want);
        for (int k = 0, i = 0; k < want; k++, i++) {
            while (!fl[i]) i++;
            CHECK(idl[0][k] == i && idl[1][k] == i);
        }
    }

    /* a support radius >= box / 2 among the guesses: nothing is computed, SPH_E_HRANGE */
    h[7] = 0.75f;
    CHECK(cudaMemcpy(d_h, h, sizeof h, cudaMemcpyHostToDevice) == cudaSuccess);
    CHECK(sph_density(ctx, NULL, -1, 64.f, 2.f, d_h, d_rho, d_om, d_ngb, d_st, &unconv) == SPH_E_HRANGE);
    /* a position outside the box: the index is unusable until rebuilt */
    float bad = 1.5f;
    CHECK(cudaMemcpy(d_pos + 3, &bad, sizeof bad, cudaMemcpyHostToDevice) == cudaSuccess);
    CHECK(sph_build_index(ctx, N, d_pos, NULL, 1.0f / N) == SPH_OK); /* asynchronous: reported by the next synchronising call */
    CHECK(sph_get_stats(ctx, &s) == SPH_E_ARG);
    CHECK(sph_destroy(ctx) == SPH_OK);
    printf("abi_smoke ok: mean rho %.4f, %lld density pairs, %lld force pairs, version %s\n", mean, (long long)s.dens_pairs,
           (long long)s.force_pairs, sph_version());
    return 0;
}
