// =====================================================================================
// lbm_inst.cu -- explicit instantiations of the launchers of lbm_launch.cuh for ONE lattice, dtype and part, chosen by
//   -DLBM_INST_Q=19|27  -DLBM_INST_T=float|double  -DLBM_INST_PART=0|1|2|3
// part 0: BGK step (collide, stream + collide, stream only) and the equilibrium initialiser; part 1: HRR form (u^ pass +
// fused step); part 2: A9 (moments, totals); part 3: the in-place AA-pattern kernels.  The build compiles the twelve objects in parallel.
// =====================================================================================
#include "lbm_launch.cuh"

namespace lbmhost {
#if LBM_INST_PART == 0
template int launch_step_bgk<LBM_INST_Q, LBM_INST_T>(lbm_ctx*, const lbm_params*, int);
template int launch_init<LBM_INST_Q, LBM_INST_T>(lbm_ctx*, const void*, const void*);
#elif LBM_INST_PART == 1
template int launch_step_hrr<LBM_INST_Q, LBM_INST_T>(lbm_ctx*, const lbm_params*, int, int);
#elif LBM_INST_PART == 2
template int launch_moments<LBM_INST_Q, LBM_INST_T>(lbm_ctx*, const lbm_params*, void*, void*);
template int launch_totals<LBM_INST_Q, LBM_INST_T>(lbm_ctx*, const lbm_params*);
#elif LBM_INST_PART == 3
template int launch_aa<LBM_INST_Q, LBM_INST_T>(lbm_ctx*, const lbm_params*, int);
#else
#error "LBM_INST_PART must be 0, 1, 2 or 3"
#endif
}  // namespace lbmhost
