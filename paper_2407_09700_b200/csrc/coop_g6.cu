// coop_g6.cu -- instantiations of the cooperative-family J/K kernel for class group 6 (coop_classes.h).
#include "coop_kernel.cuh"
#include "coop_classes.h"

namespace eri {
bool launch_coop_group6(int key, const Work& w, int nblocks, cudaStream_t s, cudaError_t* err) {
  switch (key) {
#define X(a, b, c, d, tw, nch) case a * 1000 + b * 100 + c * 10 + d: *err = launch_coop_jk<a, b, c, d, tw, nch>(w, nblocks, s); return true;
    COOP_GROUP6(X)
#undef X
    default: return false;
  }
}
}  // namespace eri
