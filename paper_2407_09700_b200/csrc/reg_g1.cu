// reg_g1.cu -- instantiations of the register-family J/K kernel for class group 1 (reg_classes.h).
#include "reg_kernel.cuh"
#include "reg_classes.h"

namespace eri {
bool launch_reg_group1(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err) {
  switch (key) {
#define X(a, b, c, d) case a * 1000 + b * 100 + c * 10 + d: *err = launch_reg_jk<a, b, c, d>(w, nblocks, s); return true;
    REG_GROUP1(X)
#undef X
    default: return false;
  }
}
}  // namespace eri
