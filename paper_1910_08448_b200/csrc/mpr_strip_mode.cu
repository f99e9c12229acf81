// mpr_strip_mode.cu -- the STRIP kernels of ONE precision mode (compile with -DMPR_STRIP_MODE=0..3).
#include "mpr_strip.cuh"

#ifndef MPR_STRIP_MODE
#error "compile with -DMPR_STRIP_MODE=<0..3>"
#endif

namespace mpr {

#define MPR_CAT2(a, b) a##b
#define MPR_CAT(a, b) MPR_CAT2(a, b)

int MPR_CAT(strip_launch_mode, MPR_STRIP_MODE)(const StripArgs& a) {
  constexpr int MODE = MPR_STRIP_MODE;
  using R = typename Traits<MODE>::real;
  return strip_launch<MODE>(*a.plan, *a.tp, a.g, a.src_index, a.src, a.dst, a.smask, a.acc, a.part, a.slots,
                            *static_cast<const ChainConst<R>*>(a.kc), a.first_sweep, a.prog, a.k, a.measure, a.stream,
                            a.nblocks_out, a.max_partials);
}

}  // namespace mpr
