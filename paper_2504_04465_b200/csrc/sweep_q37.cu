// sweep_q37.cu -- D2Q37 instantiations of the level-sweep kernels (sweep.cuh); one translation unit per
// lattice so that the instantiations compile in parallel.
#include "matrix.cuh"
#include "sweep_pipe.cuh"

namespace lbm {

int kernel_sets_q37(const KernelSet** out) {
  static const KernelSet sets[] = {
      LBM_KSET_MATRIX(37, double, LBM_BGK),
      LBM_KSET_MATRIX(37, double, LBM_RR),
      LBM_KSET_MATRIX(37, float, LBM_BGK),
      LBM_KSET_MATRIX(37, float, LBM_RR),
      LBM_KSET_PIPE(37, double, LBM_BGK, true, false),
      LBM_KSET_PIPE(37, double, LBM_BGK, true, true),
      LBM_KSET_PIPE(37, float, LBM_BGK, true, true),
      LBM_KSET_PIPE(37, double, LBM_NUMEQ, true, false),
      LBM_KSET_PIPE(37, double, LBM_NUMEQ, true, true),
      LBM_KSET_PIPE(37, float, LBM_NUMEQ, true, true)};
  *out = sets;
  return (int)(sizeof(sets) / sizeof(sets[0]));
}

}  // namespace lbm
