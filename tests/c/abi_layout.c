/* Prints size and field offsets of the structs of include/sph.h as the C compiler lays them out; the
 * test compares them with the ctypes mirror of paper_2003_10850_b200/binding.py (tests/test_library_abi.py). */
#include <stddef.h>
#include <stdio.h>

#include "sph.h"

#define F(s, f) printf(#s "." #f " %zu\n", offsetof(s, f))

int main(void)
{
    printf("sph_params %zu\n", sizeof(sph_params));
    F(sph_params, kernel); F(sph_params, box); F(sph_params, gamma); F(sph_params, alpha_visc);
    F(sph_params, count_mode); F(sph_params, max_iter); F(sph_params, group_cap); F(sph_params, group_node);
    printf("sph_stats %zu\n", sizeof(sph_stats));
    F(sph_stats, n); F(sph_stats, n_nodes); F(sph_stats, n_groups); F(sph_stats, launches);
    F(sph_stats, dens_evals); F(sph_stats, dens_candidates); F(sph_stats, dens_pairs);
    F(sph_stats, force_candidates); F(sph_stats, force_pairs);
    F(sph_stats, t_index_ms); F(sph_stats, t_density_kernel_ms); F(sph_stats, t_force_prep_ms);
    F(sph_stats, t_force_kernel_ms); F(sph_stats, node_pool_overflow);
    printf("sph_improved_params %zu\n", sizeof(sph_improved_params));
    F(sph_improved_params, alpha_min); F(sph_improved_params, alpha_max); F(sph_improved_params, decay_l);
    F(sph_improved_params, alpha_cond); F(sph_improved_params, balsara);
    printf("sph_kdk_params %zu\n", sizeof(sph_kdk_params));
    F(sph_kdk_params, dt_max); F(sph_kdk_params, n_bins); F(sph_kdk_params, courant); F(sph_kdk_params, eta);
    F(sph_kdk_params, n_ngb_target); F(sph_kdk_params, n_ngb_tol); F(sph_kdk_params, refresh_max); F(sph_kdk_params, rebuild_fraction);
    F(sph_kdk_params, grav_G); F(sph_kdk_params, grav_rs); F(sph_kdk_params, grav_rcut); F(sph_kdk_params, grav_eps); F(sph_kdk_params, grav_theta);
    printf("sph_kdk_state %zu\n", sizeof(sph_kdk_state));
    F(sph_kdk_state, pos); F(sph_kdk_state, vel); F(sph_kdk_state, u); F(sph_kdk_state, h); F(sph_kdk_state, rho);
    F(sph_kdk_state, omega); F(sph_kdk_state, ngb); F(sph_kdk_state, acc); F(sph_kdk_state, dudt); F(sph_kdk_state, vsig);
    F(sph_kdk_state, vpred); F(sph_kdk_state, upred); F(sph_kdk_state, bin); F(sph_kdk_state, tbegin); F(sph_kdk_state, active);
    printf("status %d %d %d %d %d %d %d %d\n", SPH_OK, SPH_E_ARG, SPH_E_CUDA, SPH_E_NOINDEX, SPH_E_OOM, SPH_E_INTERNAL,
           SPH_E_HRANGE, SPH_W_NOCONV);
    printf("flags %d %d %d %d\n", SPH_ST_CONVERGED, SPH_ST_BRACKET, SPH_ST_NOTCONV, SPH_ST_STALLED);
    return 0;
}
