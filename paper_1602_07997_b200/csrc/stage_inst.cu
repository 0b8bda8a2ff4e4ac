// One translation unit per (model, degree): compiled with -DDG_MODEL=<0|1> -DDG_N=<1..10>.
// Exposes the kernel entry points of kernels.cuh for that pair to dg_api.cu through a C getter.
#include "kernels.cuh"
#include "tc3_kernels.cuh"

#if !defined(DG_MODEL) || !defined(DG_N)
#error "compile with -DDG_MODEL=0|1 -DDG_N=1..10"
#endif

#define DG_CAT3_(a, b, c) a##b##_##c
#define DG_CAT3(a, b, c) DG_CAT3_(a, b, c)
#define DG_GETTER(m, n) DG_CAT3(dgk_get_stage_kernel_, m, n)

namespace {
template <int E>
const void *pick_mode(int mode) {
  if (mode == dgk::MODE_RHS) return (const void *)&dgk::stage_kernel<DG_MODEL, DG_N, E, dgk::MODE_RHS>;
  if (mode == dgk::MODE_STAGE) return (const void *)&dgk::stage_kernel<DG_MODEL, DG_N, E, dgk::MODE_STAGE>;
  return nullptr;
}
}  // namespace

// returns the __global__ function for register blocking E and mode, or NULL if not instantiated
extern "C" const void *DG_GETTER(DG_MODEL, DG_N)(int E, int mode) {
  switch (E) {
    case 1: return pick_mode<1>(mode);
    case 2: return pick_mode<2>(mode);
    case 4: return pick_mode<4>(mode);
#if DG_MODEL == 0
    case 8: return pick_mode<8>(mode);
#endif
    default: return nullptr;
  }
}

extern "C" size_t DG_CAT3(dgk_stage_smem_bytes_, DG_MODEL, DG_N)(int EB) { return dgk::Smem<DG_MODEL, DG_N>::bytes(EB); }

// pipelined warp-specialised BF16x3 tensor-core variant (tc3_kernels.cuh): every degree
extern "C" const void *DG_CAT3(dgk_get_tc3_kernel_, DG_MODEL, DG_N)(int mode) {
  if (mode == dgk::MODE_RHS) return (const void *)&dgk::tc3_stage_kernel<DG_MODEL, DG_N, dgk::MODE_RHS>;
  if (mode == dgk::MODE_STAGE) return (const void *)&dgk::tc3_stage_kernel<DG_MODEL, DG_N, dgk::MODE_STAGE>;
  return nullptr;
}
// launch geometry: what = 0 shared-memory bytes, 1 elements per batch, 2 NCH, 3 k-steps, 4 NSPLIT, 5 tile staged in
// shared memory, 6 tile slots, 7 accumulator sets, 8 A ring stages, 9 epilogue chunk width, 10 row pitch of q / res / rhs (floats)
extern "C" int DG_CAT3(dgk_tc3_info_, DG_MODEL, DG_N)(int what) {
  using C = dgk::T3<DG_MODEL, DG_N>;
  switch (what) {
    case 0: return C::SMEM;
    case 1: return C::EB;
    case 2: return C::NCH;
    case 3: return C::NSTEP;
    case 4: return C::NSPLIT;
    case 5: return C::TILE ? 1 : 0;
    case 6: return C::NQ;
    case 7: return C::NSETS;
    case 8: return C::NA;
    case 9: return C::CW;
    case 10: return C::PT;
    default: return -1;
  }
}

#ifdef DG_PROF
// role timeline of the last tc3 launch of this (model, degree): [296][23][5] long long (tc3_kernels.cuh)
extern "C" int DG_CAT3(dgk_prof_read_, DG_MODEL, DG_N)(long long *out) {
  return (int)cudaMemcpyFromSymbol(out, dgk::dg_prof_buf, sizeof(dgk::dg_prof_buf));
}
#endif
