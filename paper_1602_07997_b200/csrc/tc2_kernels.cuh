// Warp-specialised tensor-core stage kernel of libdg (sm_100a), variant 3: "tc_bf16x3".
//
// One persistent CTA per SM evaluates, batch by batch (32 acoustic / 14 elastic elements = up to 128
// element-field rows), every row of the hot path as ONE contraction on the 5th-generation tensor cores
//
//     R[row][n] = sum_k  A[row][k] * B[n][k],      row = (element, field),  n = output node
//
// with  k = (D_j, node m)  for the volume term, A = a_{f,j}[m] the pre-combined (rows a1 + a3) and
// vertex-mean shifted fields, B = D_j[n][m]   (row a2; eq. (9)-(10) P:191-204), and
// k = face node for the surface term, A = penalty terms times g^sur (rows a4, a5), B = LIFT[n][k] (row a6,
// P:206-209).  The LSRK update (row a7) is the epilogue.  Compared with tc_kernels.cuh the roles of the
// operands are transposed: the data are the M side (128 rows = TMEM lanes) and live in TENSOR MEMORY,
// written by the producer warps with tcgen05.st straight from registers (no shared-memory round trip, no
// proxy fence), the operator panel is the N side (N = Np rounded to 16, so the MMA cost follows Np
// instead of a fixed 128) and streams from L2 through a bulk-copy ring.
//
// Precision: fp32-equivalent through a BF16x3 split.  x = b1 + b2 + b3 with round-to-nearest pieces
// represents every fp32 value exactly (|b2| <= 2^-9 |x|, |b3| <= 2^-18 |x|); the operators are split from
// their fp64 values.  Six kind::f16 MMAs per 16-wide k-step: b1*b1 into the main accumulator, the five
// cross terms of order 2^-8 and 2^-16 into a second one (so that they do not add truncations to the large
// sum); the dropped terms are below 2^-26.  The two accumulators are added in fp32 in the epilogue.
//
// Warp roles (576 threads): 0-3 epilogue (TMEM -> registers -> shared-memory transpose -> coalesced
// global I/O), 4-11 producers (lane = row; pre-combination, split, tcgen05.st), 12-15 flux warps (load the
// batch's field tile, face gather + upwind penalty terms for the whole batch), 16 operator stream
// (cp.async.bulk), 17 MMA issue + TMEM allocation.  Pipelines: A ring in TMEM, B ring in shared memory,
// accumulator sets (two when 4*NC + 128 <= 512 columns), field tile, flux buffer; all mbarrier based.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "flux.cuh"
#include "kernels.cuh"
#include "tc_kernels.cuh"

namespace dgk {

constexpr int T2_THREADS = 576;
constexpr int T2_NB = 4;            // operator ring stages (shared memory)
constexpr int T2_ASTRIDE = 24;      // TMEM columns per A stage: 3 pieces x 8 columns (16 bf16)

template <int MODEL, int N>
struct T2 {
  using D = Deg<N>;
  static constexpr int NP = D::NP, NFP = D::NFP, NFACE = D::NFACE;
  static constexpr int NF = MODEL == 0 ? 4 : 9;
  static constexpr int NGEO = MODEL == 0 ? GEO_AC : GEO_EL;
  static constexpr int EB = MODEL == 0 ? 32 : 14;              // elements per batch
  static constexpr int NR = EB * NF;                           // valid rows (<= 128)
  static constexpr int NC = (NP + 15) / 16 * 16;               // MMA N (output nodes, padded)
  static constexpr int NG = (NP + 15) / 16;                    // node chunks of 16
  static constexpr int NH = (NFACE + 15) / 16;                 // face-node chunks of 16
  static constexpr int NSTEP = 3 * NG + NH;                    // k-steps of 16 per batch
  static constexpr int NSETS = (4 * NC + 128 <= 512) ? 2 : 1;  // accumulator sets
  static constexpr int ABASE = NSETS * 2 * NC;                 // first TMEM column of the A ring
  static constexpr int NA_ = (512 - ABASE) / T2_ASTRIDE;
  static constexpr int NA = NA_ > 9 ? 9 : NA_;                 // A ring stages (multiple of 3 preferred)
  static constexpr int BSTAGE = 96 * NC;                       // bytes: [3 pieces][2 kc][NC][8] bf16
  static constexpr int FS = NH * 16 + 4;                       // flux row stride (floats), = 4 or 20 mod 32
  // shared-memory carve-up (bytes)
  static constexpr int OFF_B = 0;
  static constexpr int OFF_Q = OFF_B + T2_NB * BSTAGE;
  static constexpr int OFF_FLUX = OFF_Q + ((EB * NF * NP * 4 + 15) / 16) * 16;
  static constexpr int OFF_SCR = OFF_FLUX + 128 * FS * 4;
  static constexpr int OFF_GEO = OFF_SCR + 4 * 32 * 33 * 4;
  static constexpr int OFF_NBR = OFF_GEO + EB * NGEO * 4;
  static constexpr int OFF_BAR = (OFF_NBR + EB * 8 * 4 + 15) / 16 * 16;
  static constexpr int NBAR = 2 * NA + 2 * T2_NB + 4 + 4;
  static constexpr int SMEM = OFF_BAR + NBAR * 8 + 16 + 128;   // + slack for the 128-byte alignment
  static_assert(NR <= 128 && NC <= 128, "one M tile, N <= 7");
  static_assert(NA >= 3, "A ring too small");
};

struct Tc2Params {
  StageParams s;
  const uint16_t *__restrict__ Bimg;   // [NSTEP][3][2][NC][8] bf16 operator panel image (host: build_tc2_image)
  int nbatch;
};

namespace tc {
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]^T, kind::f16 (bf16 operands, fp32 accumulate)
__device__ __forceinline__ void umma_bf16_ts(uint32_t d, uint32_t a, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(d),
      "r"(a), "l"(bdesc), "r"(idesc), "r"(acc)
      : "memory");
}
__host__ __device__ constexpr uint32_t make_idesc_bf16(int M, int Ncols) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(Ncols >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void tmem_st4(uint32_t taddr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};" ::"r"(taddr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}
// x0, x1 -> three packed bf16 pairs (b1, b2, b3), low half = x0
__device__ __forceinline__ void split3(float x0, float x1, uint32_t &p1, uint32_t &p2, uint32_t &p3) {
  p1 = pack_bf16(x0, x1);
  const float r0 = x0 - __uint_as_float(p1 << 16), r1 = x1 - __uint_as_float(p1 & 0xFFFF0000u);
  p2 = pack_bf16(r0, r1);
  const float t0 = r0 - __uint_as_float(p2 << 16), t1 = r1 - __uint_as_float(p2 & 0xFFFF0000u);
  p3 = pack_bf16(t0, t1);
}
__device__ __forceinline__ void named_bar(int id, int nthreads) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory"); }
}  // namespace tc

// ---- penalty terms of one face node (rows a4, a5): interior trace from the shared-memory field tile,
// exterior trace gathered from global memory through the compressed connectivity
template <int MODEL, int N>
__device__ __forceinline__ void flux_task(const StageParams &p, const float *s_q, const float *s_geo, const int *s_nbr,
                                          const int *s_code, int e, int j, float *F) {
  using D = Deg<N>;
  constexpr int NP = D::NP, NFP = D::NFP;
  constexpr int NF = MODEL == 0 ? 4 : 9, NGEO = MODEL == 0 ? GEO_AC : GEO_EL;
  const int f = j / NFP, i = j - f * NFP;
  const float *g = s_geo + e * NGEO;
  const int nm = p.fmask[j];
  const int nb = s_nbr[e * 4 + f];
  const float *qm = s_q + (e * NF) * NP + nm;
  if (MODEL == 0) {
    const float *fg = g + 12 + 5 * f;
    const float nx = fg[0], ny = fg[1], nz = fg[2];
    const float pm = qm[0], vxm = qm[NP], vym = qm[2 * NP], vzm = qm[3 * NP];
    float dp, dvn;
    if (nb >= 0) {
      const int nn = p.nbrnode[(f * 24 + s_code[e * 4 + f]) * NFP + i];
      const float *qp = p.q_in + ((size_t)nb * NF) * NP + nn;
      dp = __ldg(qp) - pm;
      dvn = (__ldg(qp + NP) - vxm) * nx + (__ldg(qp + 2 * NP) - vym) * ny + (__ldg(qp + 3 * NP) - vzm) * nz;
    } else {
      acoustic_boundary_jump(nb, pm, vxm * nx + vym * ny + vzm * nz, dp, dvn);
    }
    const float4 P = acoustic_penalty(g, fg, dp, dvn);
    F[0] = P.x; F[1] = P.y; F[2] = P.z; F[3] = P.w;
  } else {
    const float *fg = g + 16 + 8 * f;
    const float nx = fg[0], ny = fg[1], nz = fg[2];
    float um[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) um[c] = qm[c * NP];
    float Tmx, Tmy, Tmz;
    traction(um, nx, ny, nz, Tmx, Tmy, Tmz);
    float dv[3], dT[3];
    if (nb >= 0) {
      const int nn = p.nbrnode[(f * 24 + s_code[e * 4 + f]) * NFP + i];
      const float *qp = p.q_in + ((size_t)nb * NF) * NP + nn;
      float up[9];
#pragma unroll
      for (int c = 0; c < 9; ++c) up[c] = __ldg(qp + c * NP);
      float Tpx, Tpy, Tpz;
      traction(up, nx, ny, nz, Tpx, Tpy, Tpz);
      dv[0] = up[0] - um[0]; dv[1] = up[1] - um[1]; dv[2] = up[2] - um[2];
      dT[0] = Tpx - Tmx; dT[1] = Tpy - Tmy; dT[2] = Tpz - Tmz;
    } else {
      elastic_boundary_jump(nb, um, Tmx, Tmy, Tmz, nx, ny, nz, dv, dT);
    }
    elastic_penalty(g, fg, dv, dT, F);
  }
}

// ---- per-row pre-combination coefficients (rows a1 + a3):  a_j = sum_i cf[j][i] * (u_src[i] - mean_i)
template <int MODEL>
__device__ __forceinline__ void row_coefficients(const float *__restrict__ g, int f, float cf[3][3], int src[3], int &nsrc) {
  float G[9];
#pragma unroll
  for (int i = 0; i < 9; ++i) G[i] = __ldg(g + i);
#pragma unroll
  for (int j = 0; j < 3; ++j)
#pragma unroll
    for (int i = 0; i < 3; ++i) cf[j][i] = 0.f;
  src[0] = src[1] = src[2] = 0;
  if (MODEL == 0) {
    const float kap = __ldg(g + 9), irho = __ldg(g + 10);
    if (f == 0) {                   // eq. (5): r_p = -kappa sum_j D_j (sum_i g_ij v_i)
      nsrc = 3;
      src[0] = 1; src[1] = 2; src[2] = 3;
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int i = 0; i < 3; ++i) cf[j][i] = -kap * G[3 * i + j];
    } else {                        // eq. (6): r_vi = -(1/rho) sum_j g_ij D_j p
      nsrc = 1;
#pragma unroll
      for (int j = 0; j < 3; ++j) cf[j][0] = -irho * G[3 * (f - 1) + j];
    }
  } else {
    const float irho = __ldg(g + 9), lam = __ldg(g + 10), mu = __ldg(g + 11);
    nsrc = 3;
    if (f < 3) {                    // r_vi = (1/rho) sum_j D_j (sum_m g_mj sigma_im)
      const int row[3][3] = {{3, 6, 7}, {6, 4, 8}, {7, 8, 5}};
#pragma unroll
      for (int m = 0; m < 3; ++m) src[m] = row[f][m];
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int m = 0; m < 3; ++m) cf[j][m] = irho * G[3 * m + j];
    } else {                        // PAPER.md:158 (reading Q6): lambda delta_ab div v + mu (d_b v_a + d_a v_b)
      src[0] = 0; src[1] = 1; src[2] = 2;
      const int a = f < 6 ? f - 3 : (f == 8 ? 1 : 0);
      const int bb = f < 6 ? f - 3 : (f == 6 ? 1 : 2);
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        if (f < 6) {
#pragma unroll
          for (int i = 0; i < 3; ++i) cf[j][i] = lam * G[3 * i + j];
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          if (i == a) cf[j][i] += mu * G[3 * bb + j];
          if (i == bb) cf[j][i] += mu * G[3 * a + j];
        }
      }
    }
  }
}

// ---- the kernel ------------------------------------------------------------------------------------
template <int MODEL, int N, int MODE>
__global__ void __launch_bounds__(T2_THREADS, 1) tc2_stage_kernel(const Tc2Params P) {
  using C = T2<MODEL, N>;
  constexpr int NP = C::NP, NFACE = C::NFACE, NF = C::NF, NGEO = C::NGEO, EB = C::EB, NC = C::NC;
  constexpr int NA = C::NA, NB = T2_NB;
  const StageParams &p = P.s;

  extern __shared__ unsigned char smem_raw[];
  unsigned char *sm = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~(uintptr_t)127);
  unsigned char *sB = sm + C::OFF_B;                               // [NB][3][2][NC][8] bf16
  float *s_q = reinterpret_cast<float *>(sm + C::OFF_Q);           // [EB][NF][NP] field tile of the batch
  float *s_flux = reinterpret_cast<float *>(sm + C::OFF_FLUX);     // [128][FS] penalty terms of the batch
  float *s_scr = reinterpret_cast<float *>(sm + C::OFF_SCR);       // [4][32][33] epilogue transpose
  float *s_geo = reinterpret_cast<float *>(sm + C::OFF_GEO);       // [EB][NGEO]
  int *s_nbr = reinterpret_cast<int *>(sm + C::OFF_NBR);           // [EB][4]
  int *s_code = s_nbr + EB * 4;                                    // [EB][4]
  uint64_t *bars = reinterpret_cast<uint64_t *>(sm + C::OFF_BAR);
  uint32_t *s_tmem = reinterpret_cast<uint32_t *>(bars + C::NBAR);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t bar0 = tc::smem_u32(bars);
  auto fullA = [&](int t) { return bar0 + 8u * t; };
  auto emptyA = [&](int t) { return bar0 + 8u * (NA + t); };
  auto fullB = [&](int t) { return bar0 + 8u * (2 * NA + t); };
  auto emptyB = [&](int t) { return bar0 + 8u * (2 * NA + NB + t); };
  auto accFull = [&](int t) { return bar0 + 8u * (2 * NA + 2 * NB + t); };
  auto accEmpty = [&](int t) { return bar0 + 8u * (2 * NA + 2 * NB + 2 + t); };
  const uint32_t qFull = bar0 + 8u * (2 * NA + 2 * NB + 4), qEmpty = qFull + 8, fluxFull = qFull + 16, fluxEmpty = qFull + 24;

  if (warp == 17) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(s_tmem)), "n"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid == 0) {
    for (int t = 0; t < NA; ++t) { tc::mbar_init(fullA(t), 8); tc::mbar_init(emptyA(t), 1); }
    for (int t = 0; t < NB; ++t) { tc::mbar_init(fullB(t), 1); tc::mbar_init(emptyB(t), 1); }
    for (int t = 0; t < 2; ++t) { tc::mbar_init(accFull(t), 1); tc::mbar_init(accEmpty(t), 4); }
    tc::mbar_init(qFull, 4); tc::mbar_init(qEmpty, 12); tc::mbar_init(fluxFull, 4); tc::mbar_init(fluxEmpty, 8);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tm = *s_tmem;

  if (warp < 4) {
    // =================================================== epilogue: LSRK update (row a7), coalesced I/O
    const int qd = warp;
    float *scr = s_scr + warp * (32 * 33);
    constexpr int NCH = (NP + 31) / 32;
    int it = 0;
    for (int b = blockIdx.x; b < P.nbatch; b += gridDim.x, ++it) {
      const int k0 = b * EB;
      const int nrows = min(EB, p.K - k0) * NF;
      const int set = C::NSETS == 2 ? (it & 1) : 0, use = C::NSETS == 2 ? (it >> 1) : it;
      tc::mbar_wait(accFull(set), use & 1);
      tc::tc_fence_after();
      const uint32_t t0 = tm + ((uint32_t)(qd * 32) << 16) + set * 2 * NC;
#pragma unroll 1
      for (int ch = 0; ch < NCH; ++ch) {
        const int c0 = ch * 32;
        uint32_t vm[32], vs[32];
        tc::tmem_ld32(t0 + c0, vm);
        tc::tmem_ld32(t0 + NC + c0, vs);
        if (ch == NCH - 1) {             // accumulators drained: the MMA warp may start the next batch on this set
          tc::tc_fence_before();
          __syncwarp();
          if (lane == 0) tc::mbar_arrive(accEmpty(set));
        }
#pragma unroll
        for (int j = 0; j < 32; ++j) scr[lane * 33 + j] = __uint_as_float(vm[j]) + __uint_as_float(vs[j]);
        __syncwarp();
        const int n = c0 + lane;
        const int rmax = min(32, nrows - qd * 32);
        if (n < NP) {
          const size_t base = ((size_t)k0 * NF + qd * 32) * NP + n;
#pragma unroll 4
          for (int rr = 0; rr < rmax; ++rr) {
            const float r = scr[rr * 33 + lane];
            const size_t idx = base + (size_t)rr * NP;
            if (MODE == MODE_RHS) {
              p.rhs[idx] = r;
            } else {
              float rs = p.dt * r;
              if (p.a != 0.f) rs = fmaf(p.a, p.res[idx], rs);
              p.res[idx] = rs;
              p.q_out[idx] = fmaf(p.b, rs, __ldg(p.q_in + idx));
            }
          }
        }
        __syncwarp();
      }
    }
  } else if (warp < 12) {
    // =================================================== producers: rows a1 + a3, BF16x3 split, tcgen05.st
    const int pw = warp - 4, qd = pw & 3, half = pw >> 2;
    const int r = qd * 32 + lane;                      // row = (element e, field f)
    const int e = r / NF, f = r - e * NF;
    const uint32_t trow = tm + ((uint32_t)(qd * 32) << 16) + C::ABASE + 4 * half;
    constexpr bool VEC4 = (NP % 4) == 0;
    int slot = 0;
    uint32_t phase = 0;
    auto emit = [&](const float *a) {                  // 8 values of this row for one k-step -> TMEM
      uint32_t p1[4], p2[4], p3[4];
#pragma unroll
      for (int t = 0; t < 4; ++t) tc::split3(a[2 * t], a[2 * t + 1], p1[t], p2[t], p3[t]);
      tc::mbar_wait(emptyA(slot), phase ^ 1);
      tc::tc_fence_after();
      const uint32_t ta = trow + slot * T2_ASTRIDE;
      tc::tmem_st4(ta, p1[0], p1[1], p1[2], p1[3]);
      tc::tmem_st4(ta + 8, p2[0], p2[1], p2[2], p2[3]);
      tc::tmem_st4(ta + 16, p3[0], p3[1], p3[2], p3[3]);
      tc::tmem_st_wait();
      tc::tc_fence_before();
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(fullA(slot));
      if (++slot == NA) { slot = 0; phase ^= 1; }
    };
    int it = 0;
    for (int b = blockIdx.x; b < P.nbatch; b += gridDim.x, ++it) {
      const int k0 = b * EB;
      const int nvalid = min(EB, p.K - k0);
      const bool valid = r < C::NR && e < nvalid;
      float cf[3][3];
      int src[3] = {0, 0, 0}, nsrc = 0;
      if (valid) {
        row_coefficients<MODEL>(p.geo + (size_t)(k0 + e) * NGEO, f, cf, src, nsrc);
      } else {
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
          for (int i = 0; i < 3; ++i) cf[j][i] = 0.f;
      }
      tc::mbar_wait(qFull, it & 1);
      const float *sp[3];
      float mean[3];
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        sp[i] = s_q + (e * NF + src[i]) * NP;
        // mean of the four vertex values: D_j 1 = 0, so the shift is exact and removes the cancellation
        mean[i] = (valid && i < nsrc) ? 0.25f * ((sp[i][0] + sp[i][N]) + (sp[i][C::NFP - 1] + sp[i][NP - 1])) : 0.f;
      }
#pragma unroll 1
      for (int g = 0; g < C::NG; ++g) {
        const int m0 = 16 * g + 8 * half;
        float u[3][8];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          if (valid && i < nsrc && m0 < NP) {
            if (VEC4) {
#pragma unroll
              for (int h4 = 0; h4 < 2; ++h4) {
                if (m0 + 4 * h4 < NP) {
                  const float4 v = *reinterpret_cast<const float4 *>(sp[i] + m0 + 4 * h4);
                  u[i][4 * h4 + 0] = v.x - mean[i]; u[i][4 * h4 + 1] = v.y - mean[i];
                  u[i][4 * h4 + 2] = v.z - mean[i]; u[i][4 * h4 + 3] = v.w - mean[i];
                } else {
                  u[i][4 * h4 + 0] = u[i][4 * h4 + 1] = u[i][4 * h4 + 2] = u[i][4 * h4 + 3] = 0.f;
                }
              }
            } else {
#pragma unroll
              for (int t = 0; t < 8; ++t) u[i][t] = (m0 + t < NP) ? sp[i][m0 + t] - mean[i] : 0.f;
            }
          } else {
#pragma unroll
            for (int t = 0; t < 8; ++t) u[i][t] = 0.f;
          }
        }
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          float a[8];
#pragma unroll
          for (int t = 0; t < 8; ++t) a[t] = cf[j][0] * u[0][t] + cf[j][1] * u[1][t] + cf[j][2] * u[2][t];
          emit(a);
        }
      }
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(qEmpty);          // this warp no longer reads the field tile
      tc::mbar_wait(fluxFull, it & 1);
#pragma unroll 1
      for (int h = 0; h < C::NH; ++h) {
        const int j0 = 16 * h + 8 * half;
        float a[8];
        if (valid) {
          const float4 v0 = *reinterpret_cast<const float4 *>(s_flux + r * C::FS + j0);
          const float4 v1 = *reinterpret_cast<const float4 *>(s_flux + r * C::FS + j0 + 4);
          a[0] = v0.x; a[1] = v0.y; a[2] = v0.z; a[3] = v0.w; a[4] = v1.x; a[5] = v1.y; a[6] = v1.z; a[7] = v1.w;
#pragma unroll
          for (int t = 0; t < 8; ++t) a[t] = (j0 + t < NFACE) ? a[t] : 0.f;
        } else {
#pragma unroll
          for (int t = 0; t < 8; ++t) a[t] = 0.f;
        }
        emit(a);
      }
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(fluxEmpty);
    }
  } else if (warp < 16) {
    // =================================================== flux warps: field tile load, rows a4 + a5
    const int ft = tid - 384;
    int it = 0;
    for (int b = blockIdx.x; b < P.nbatch; b += gridDim.x, ++it) {
      const int k0 = b * EB;
      const int nvalid = min(EB, p.K - k0);
      tc::mbar_wait(qEmpty, (it & 1) ^ 1);             // producers and flux warps are done with the previous tile
      const float *src = p.q_in + (size_t)k0 * NF * NP;
      const uint32_t bytes = (uint32_t)nvalid * NF * NP * 4u;
      if (((reinterpret_cast<uintptr_t>(src) | bytes) & 15) == 0) {
        if (ft == 0) {
          tc::mbar_expect_tx(qFull, bytes);
          tc::bulk_g2s(tc::smem_u32(s_q), src, bytes, qFull);
        } else if (lane == 0) {
          tc::mbar_arrive(qFull);
        }
      } else {                                          // misaligned run (odd Np): cooperative copy
        for (int x = ft; x < nvalid * NF * NP; x += 128) s_q[x] = __ldg(src + x);
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(qFull);
      }
      for (int x = ft; x < nvalid * NGEO; x += 128) s_geo[x] = __ldg(p.geo + (size_t)k0 * NGEO + x);
      for (int x = ft; x < nvalid * 4; x += 128) {
        s_nbr[x] = __ldg(p.nbr + (size_t)k0 * 4 + x);
        s_code[x] = (int)__ldg(p.fcode + (size_t)k0 * 4 + x);
      }
      tc::named_bar(1, 128);
      tc::mbar_wait(qFull, it & 1);
      tc::mbar_wait(fluxEmpty, (it & 1) ^ 1);          // producers have consumed the previous batch's penalty terms
      for (int t = ft; t < nvalid * NFACE; t += 128) {
        const int e = t / NFACE, j = t - e * NFACE;
        float F[NF];
        flux_task<MODEL, N>(p, s_q, s_geo, s_nbr, s_code, e, j, F);
#pragma unroll
        for (int f = 0; f < NF; ++f) s_flux[(e * NF + f) * C::FS + j] = F[f];
      }
      __syncwarp();
      if (lane == 0) {
        tc::mbar_arrive(fluxFull);
        tc::mbar_arrive(qEmpty);
      }
    }
  } else if (warp == 16) {
    // =================================================== operator stream (rows a2, a6): L2 -> shared-memory ring
    if (lane == 0) {
      int slot = 0;
      uint32_t phase = 0;
      for (int b = blockIdx.x; b < P.nbatch; b += gridDim.x) {
        for (int st = 0; st < C::NSTEP; ++st) {
          tc::mbar_wait(emptyB(slot), phase ^ 1);
          tc::mbar_expect_tx(fullB(slot), C::BSTAGE);
          tc::bulk_g2s(tc::smem_u32(sB + slot * C::BSTAGE), P.Bimg + (size_t)st * (C::BSTAGE / 2), C::BSTAGE, fullB(slot));
          if (++slot == NB) { slot = 0; phase ^= 1; }
        }
      }
    }
  } else {
    // =================================================== MMA issue: six BF16 MMAs per k-step
    if (lane == 0) {
      constexpr uint32_t IDESC = tc::make_idesc_bf16(128, NC);
      const uint64_t descB0 = tc::make_desc(tc::smem_u32(sB), NC * 16, 128);
      int sa = 0, sb = 0, it = 0;
      uint32_t pa = 0, pb = 0;
      for (int b = blockIdx.x; b < P.nbatch; b += gridDim.x, ++it) {
        const int set = C::NSETS == 2 ? (it & 1) : 0, use = C::NSETS == 2 ? (it >> 1) : it;
        tc::mbar_wait(accEmpty(set), (use & 1) ^ 1);
        tc::tc_fence_after();
        const uint32_t d0 = tm + set * 2 * NC, d1 = d0 + NC;
        for (int st = 0; st < C::NSTEP; ++st) {
          tc::mbar_wait(fullA(sa), pa);
          tc::mbar_wait(fullB(sb), pb);
          tc::tc_fence_after();
          const uint32_t a1 = tm + C::ABASE + sa * T2_ASTRIDE, a2 = a1 + 8, a3 = a1 + 16;
          const uint64_t b1 = descB0 + (uint64_t)(sb * 6 * NC), b2 = b1 + 2 * NC, b3 = b2 + 2 * NC;
          const uint32_t acc = st > 0 ? 1u : 0u;
          tc::umma_bf16_ts(d1, a2, b1, IDESC, acc);    // cross terms, orders 2^-8 and 2^-16
          tc::umma_bf16_ts(d1, a1, b2, IDESC, 1u);
          tc::umma_bf16_ts(d1, a3, b1, IDESC, 1u);
          tc::umma_bf16_ts(d1, a2, b2, IDESC, 1u);
          tc::umma_bf16_ts(d1, a1, b3, IDESC, 1u);
          tc::umma_bf16_ts(d0, a1, b1, IDESC, acc);    // leading term
          tc::umma_commit(emptyA(sa));
          tc::umma_commit(emptyB(sb));
          if (++sa == NA) { sa = 0; pa ^= 1; }
          if (++sb == NB) { sb = 0; pb ^= 1; }
        }
        tc::umma_commit(accFull(set));
      }
    }
  }

  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  if (warp == 17) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm), "n"(512) : "memory");
  }
}

}  // namespace dgk
