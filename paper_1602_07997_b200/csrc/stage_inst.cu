// One translation unit per (model, degree): compiled with -DDG_MODEL=<0|1> -DDG_N=<1..10>.
// Exposes the kernel entry points of kernels.cuh for that pair to dg_api.cu through a C getter.
#include "kernels.cuh"
#include "tc3_kernels.cuh"
#include "epk_kernels.cuh"
#include "iface_kernels.cuh"
#include "rpt_kernels.cuh"

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
  if (mode == dgk::MODE_AB3) return (const void *)&dgk::stage_kernel<DG_MODEL, DG_N, E, dgk::MODE_AB3>;
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
  if (mode == dgk::MODE_AB3) return (const void *)&dgk::tc3_stage_kernel<DG_MODEL, DG_N, dgk::MODE_AB3>;
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

// interface-centric surface kernel (iface_kernels.cuh)
extern "C" const void *DG_CAT3(dgk_get_iface_kernel_, DG_MODEL, DG_N)(void) {
  return (const void *)&dgk::iface_flux_kernel<DG_MODEL, DG_N>;
}

#ifdef DG_PROF
// role timeline of the last tc3 launch of this (model, degree): [296][23][5] long long (tc3_kernels.cuh)
extern "C" int DG_CAT3(dgk_prof_read_, DG_MODEL, DG_N)(long long *out) {
  return (int)cudaMemcpyFromSymbol(out, dgk::dg_prof_buf, sizeof(dgk::dg_prof_buf));
}
#endif

// element-per-thread kernel (epk_kernels.cuh): acoustic N = 1, 2 and elastic N = 1; NULL otherwise
#define DG_HAS_EPK (DG_N == 1 || (DG_N == 2 && DG_MODEL == 0))
extern "C" const void *DG_CAT3(dgk_get_epk_kernel_, DG_MODEL, DG_N)(int mode) {
#if DG_HAS_EPK
  if (mode == dgk::MODE_RHS) return (const void *)&dgk::epk_stage_kernel<DG_MODEL, DG_N, dgk::MODE_RHS>;
  if (mode == dgk::MODE_STAGE) return (const void *)&dgk::epk_stage_kernel<DG_MODEL, DG_N, dgk::MODE_STAGE>;
  if (mode == dgk::MODE_AB3) return (const void *)&dgk::epk_stage_kernel<DG_MODEL, DG_N, dgk::MODE_AB3>;
#endif
  (void)mode;
  return nullptr;
}
// uploads the reference operators into this translation unit's constant memory: D [3][Np][Np], L [Np][4Nfp] row-major,
// nbrnode [4][24][Nfp]; fmask [4][Nfp] must equal the kernel's compile-time table.  Returns 0, a cudaError_t, or -1
// if the face masks differ.
extern "C" int DG_CAT3(dgk_epk_upload_, DG_MODEL, DG_N)(const float *D, const float *L, const unsigned short *nbrnode, const int *fmask) {
#if DG_HAS_EPK
  using Dg = dgk::Deg<DG_N>;
  constexpr dgk::EpkFmask<DG_N> FM{};
  for (int i = 0; i < 4 * Dg::NFP; ++i)
    if (fmask[i] != FM.v[i]) return -1;
  cudaError_t e = cudaMemcpyToSymbol(dgk::c_epk_D, D, sizeof(float) * 3 * Dg::NP * Dg::NP);
  if (e == cudaSuccess) e = cudaMemcpyToSymbol(dgk::c_epk_L, L, sizeof(float) * Dg::NP * Dg::NFACE);
  {   // the same operators with the output node fastest (FFMA2 operand pairs)
    float Dt[3 * Dg::NP * Dg::NP], Lt[Dg::NFACE * Dg::NP];
    for (int j = 0; j < 3; ++j)
      for (int n = 0; n < Dg::NP; ++n)
        for (int m = 0; m < Dg::NP; ++m) Dt[(j * Dg::NP + m) * Dg::NP + n] = D[(j * Dg::NP + n) * Dg::NP + m];
    for (int n = 0; n < Dg::NP; ++n)
      for (int j = 0; j < Dg::NFACE; ++j) Lt[j * Dg::NP + n] = L[n * Dg::NFACE + j];
    if (e == cudaSuccess) e = cudaMemcpyToSymbol(dgk::c_epk_Dt, Dt, sizeof(Dt));
    if (e == cudaSuccess) e = cudaMemcpyToSymbol(dgk::c_epk_Lt, Lt, sizeof(Lt));
  }
  if (e == cudaSuccess) e = cudaMemcpyToSymbol(dgk::c_epk_nbrnode, nbrnode, sizeof(unsigned short) * 4 * 24 * Dg::NFP);
  return (int)e;
#else
  (void)D; (void)L; (void)nbrnode; (void)fmask;
  return -2;
#endif
}

// row-per-thread kernel (rpt_kernels.cuh): N <= 3; NULL otherwise
#define DG_HAS_RPT (DG_N <= 3)
extern "C" const void *DG_CAT3(dgk_get_rpt_kernel_, DG_MODEL, DG_N)(int mode) {
#if DG_HAS_RPT
  if (mode == dgk::MODE_RHS) return (const void *)&dgk::rpt_stage_kernel<DG_MODEL, DG_N, dgk::MODE_RHS>;
  if (mode == dgk::MODE_STAGE) return (const void *)&dgk::rpt_stage_kernel<DG_MODEL, DG_N, dgk::MODE_STAGE>;
  if (mode == dgk::MODE_AB3) return (const void *)&dgk::rpt_stage_kernel<DG_MODEL, DG_N, dgk::MODE_AB3>;
#endif
  (void)mode;
  return nullptr;
}
// what = 0 threads per CTA, 1 elements per CTA
extern "C" int DG_CAT3(dgk_rpt_info_, DG_MODEL, DG_N)(int what) {
#if DG_HAS_RPT
  using C = dgk::Rpt<DG_MODEL, DG_N>;
  return what == 0 ? C::WARPS * 32 : (what == 1 ? C::EPC : -1);
#else
  (void)what;
  return -1;
#endif
}
// uploads the operators into this translation unit's constant memory: DT [m][j][n] = D_j[n][m], LT [j][n] = LIFT[n][j]
extern "C" int DG_CAT3(dgk_rpt_upload_, DG_MODEL, DG_N)(const float *DT, const float *LT) {
#if DG_HAS_RPT
  using Dg = dgk::Deg<DG_N>;
  cudaError_t e = cudaMemcpyToSymbol(dgk::c_rpt_D, DT, sizeof(float) * 3 * Dg::NP * Dg::NP);
  if (e == cudaSuccess) e = cudaMemcpyToSymbol(dgk::c_rpt_L, LT, sizeof(float) * Dg::NP * Dg::NFACE);
  return (int)e;
#else
  (void)DT; (void)LT;
  return -2;
#endif
}
