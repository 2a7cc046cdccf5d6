// sweep_q9.cu -- D2Q9 instantiations of the level-sweep kernels (sweep.cuh); one translation unit per
// lattice so that the instantiations compile in parallel.
#include "matrix.cuh"

namespace lbm {

int kernel_sets_q9(const KernelSet** out) {
  static const KernelSet sets[] = {
      LBM_KSET_MATRIX(9, double, LBM_BGK),
      LBM_KSET_MATRIX(9, double, LBM_RR),
      LBM_KSET_MATRIX(9, float, LBM_BGK),
      LBM_KSET_MATRIX(9, float, LBM_RR)};
  *out = sets;
  return (int)(sizeof(sets) / sizeof(sets[0]));
}

}  // namespace lbm
