// Tensor-core stage kernel of libdg (sm_100a): the whole hot path of one RK stage as ONE batched
// contraction on the 5th-generation tensor cores (tcgen05.mma kind::tf32, accumulators in TMEM),
// in fp32-equivalent precision through a 3xTF32 split.
//
// Formulation ("pre-combination only").  All per-element coefficients of eq. (5)-(6) / PAPER.md:156-158
// (g^vol, rho, kappa / lambda, mu) are constant over an element and the D_j are linear, so for every
// field f of element k
//     r_f = [D_r D_s D_t LIFT] * [a_{f,r}; a_{f,s}; a_{f,t}; F_f]
// with a_{f,j} a node-wise linear combination of the (vertex-mean shifted) fields (rows a1+a3 folded
// into the operand) and F_f the penalty terms times g^sur (rows a4, a5).  The operator panel
// (Np x (3Np+4Nfp), rows a2+a6) is the A operand, shared by all elements and streamed from L2 by bulk
// async copies; the B operand (K x 128 columns = 32 acoustic / 14 elastic elements x fields) is
// produced on the fly into shared memory in the UMMA no-swizzle K-major core-matrix layout; the LSRK
// update (row a7) is the epilogue straight out of TMEM with coalesced stores (node = TMEM lane).
//
// Precision.  kind::tf32 reads only the top 19 bits of each operand and the tensor core truncates
// (round toward zero) when it adds into the fp32 accumulator (measured on B200).  Both
// operands are therefore split x = hi + lo with round-to-nearest (hi, lo exactly representable in TF32;
// hi + lo carries ~22 mantissa bits) and three MMAs are issued per k-step: hi*hi into the main
// accumulator, lo*hi and hi*lo into a second accumulator (their magnitude is 2^-11 of the main one,
// so adding them there would cost one truncation of the large sum per MMA); the two are added in fp32
// registers in the epilogue.
//
// Pipeline per CTA (256 threads, 2 CTAs per SM so that one CTA's epilogue overlaps the other's MMAs):
// two shared-memory stages of 3 k-steps (24 k) each; thread 0 issues the bulk copy of the operator
// slice and, after the CTA has produced the B slice, the 9 MMAs of the stage, which run asynchronously
// while the CTA produces the next slice; tcgen05.commit -> mbarrier frees the stage.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "flux.cuh"
#include "kernels.cuh"

namespace dgk {

constexpr int TC_NCOL = 128;                                   // B columns (= MMA N) per batch
constexpr int TC_THREADS = 256;
constexpr int TC_STAGE_K = 3;                                  // k-steps (of 8) per shared-memory stage
constexpr int TC_TILE_FLOATS = 128 * 8;                        // one k-step of one split: 128 rows x 8 k
constexpr int TC_A_STAGE_FLOATS = TC_STAGE_K * 2 * TC_TILE_FLOATS;   // [kstep][hi|lo][k4][row][4]
constexpr int TC_B_STAGE_FLOATS = 2 * TC_STAGE_K * TC_TILE_FLOATS;   // [hi|lo][kstep][k4][col][4]
constexpr int TC_FLUX_STRIDE = 28;                             // floats per column of the flux scratch (24 + pad)
constexpr int TC_FLUX_FLOATS = TC_NCOL * TC_FLUX_STRIDE;
constexpr int TC_SMEM_BYTES = (2 * (TC_A_STAGE_FLOATS + TC_B_STAGE_FLOATS) + TC_FLUX_FLOATS) * 4 + 128;
constexpr int TC_TMEM_COLS = 256;                              // main [0,128) + small-terms [128,256)

struct TcParams {
  StageParams s;
  const float *__restrict__ Aimg;    // [nstage][TC_A_STAGE_FLOATS] operator panel image (host_setup: build_tc_image)
  int nbatch;
};

template <int N>
struct TcDeg {
  static constexpr int NG = (Deg<N>::NP + 7) / 8;              // node stages (8 nodes x 3 operators)
  static constexpr int NFS = (Deg<N>::NFACE + 23) / 24;        // face stages (24 face nodes)
  static constexpr int NSTAGE = NG + NFS;
};

// ---- PTX wrappers ---------------------------------------------------------------------------------
namespace tc {
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// shared-memory matrix descriptor, no swizzle, K-major: core matrix = 8 rows x 16 B stored as 128
// contiguous bytes; LBO = byte distance between core matrices adjacent in K, SBO = between 8-row groups
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((saddr >> 4) & 0x3FFF) | ((uint64_t)((lbo >> 4) & 0x3FFF) << 16) | ((uint64_t)((sbo >> 4) & 0x3FFF) << 32) |
         ((uint64_t)1 << 46);
}
// instruction descriptor: D fp32, A/B tf32, both K-major, dense
__host__ __device__ constexpr uint32_t make_idesc(int M, int Ncols) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(Ncols >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void umma_tf32(uint32_t taddr, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(taddr),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t cnt) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(cnt) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred P1;\n\tLAB_WAIT:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1, %2;\n\t"
      "@P1 bra DONE;\n\tbra LAB_WAIT;\n\tDONE:\n\t}\n" ::"r"(bar),
      "r"(parity), "r"(0x989680)       // suspend-time hint: the warp sleeps in hardware instead of spinning on issue slots
      : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// 1-D bulk async copy global -> shared, completion counted in bytes on an mbarrier (TMA engine)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(__cvta_generic_to_global(src)), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// 32 lanes x 32 columns of TMEM -> 32 registers per thread (thread = lane of the warp's quadrant); the wait is
// part of the same statement so that no use of the registers can be scheduled before it
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t *v) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, "
      "[%32];\n\ttcgen05.wait::ld.sync.aligned;\n"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
        "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
        "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr)
      : "memory");
}
// round to nearest TF32 (10 explicit mantissa bits); the result is an fp32 with 13 zero low bits
__device__ __forceinline__ float tf32_rna(float x) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
  return __uint_as_float(r);
}
__device__ __forceinline__ void split_store(float *hi_dst, float *lo_dst, float a, float b, float c, float d) {
  float4 h, l;
  h.x = tf32_rna(a); l.x = tf32_rna(a - h.x);
  h.y = tf32_rna(b); l.y = tf32_rna(b - h.y);
  h.z = tf32_rna(c); l.z = tf32_rna(c - h.z);
  h.w = tf32_rna(d); l.w = tf32_rna(d - h.w);
  *reinterpret_cast<float4 *>(hi_dst) = h;
  *reinterpret_cast<float4 *>(lo_dst) = l;
}
}  // namespace tc

// ---- penalty terms of one face node, read from global memory (rows a4, a5) -------------------------
template <int MODEL, int N>
__device__ __forceinline__ void face_node_flux(const StageParams &p, int kk, int j, float *F) {
  using D = Deg<N>;
  constexpr int NP = D::NP, NFP = D::NFP;
  constexpr int NF = MODEL == 0 ? 4 : 9, NGEO = MODEL == 0 ? GEO_AC : GEO_EL;
  const int f = j / NFP, i = j - f * NFP;
  const float *g = p.geo + (size_t)kk * NGEO;
  const int nm = p.fmask[j];
  const int nb = __ldg(p.nbr + (size_t)kk * 4 + f);
  const float *qm = p.q_in + ((size_t)kk * NF) * NP + nm;
  if (MODEL == 0) {
    const float *fg = g + 12 + 5 * f;
    const float nx = __ldg(fg), ny = __ldg(fg + 1), nz = __ldg(fg + 2);
    const float pm = __ldg(qm), vxm = __ldg(qm + NP), vym = __ldg(qm + 2 * NP), vzm = __ldg(qm + 3 * NP);
    float dp, dvn;
    if (nb >= 0) {
      const int nn = p.nbrnode[(f * 24 + (int)__ldg(p.fcode + (size_t)kk * 4 + f)) * NFP + i];
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
    const float nx = __ldg(fg), ny = __ldg(fg + 1), nz = __ldg(fg + 2);
    float um[9];
#pragma unroll
    for (int c = 0; c < 9; ++c) um[c] = __ldg(qm + c * NP);
    float Tmx, Tmy, Tmz;
    traction(um, nx, ny, nz, Tmx, Tmy, Tmz);
    float dv[3], dT[3];
    if (nb >= 0) {
      const int nn = p.nbrnode[(f * 24 + (int)__ldg(p.fcode + (size_t)kk * 4 + f)) * NFP + i];
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

// ---- the kernel ------------------------------------------------------------------------------------
template <int MODEL, int N, int MODE>
__global__ void __launch_bounds__(TC_THREADS, 2) tc_stage_kernel(const TcParams P) {
  using D = Deg<N>;
  using T = TcDeg<N>;
  constexpr int NP = D::NP, NFP = D::NFP, NFACE = D::NFACE;
  constexpr int NF = MODEL == 0 ? 4 : 9, NGEO = MODEL == 0 ? GEO_AC : GEO_EL;
  constexpr int EB = TC_NCOL / NF;                 // elements per batch: 32 acoustic, 14 elastic
  constexpr bool VEC4 = (NP % 4) == 0;             // 16-byte aligned node quads
  static_assert(NP <= 128, "one M tile: Np <= 128");
  const StageParams &p = P.s;

  extern __shared__ unsigned char smem_raw[];
  float *smem = reinterpret_cast<float *>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~(uintptr_t)127);
  float *sA = smem;                                        // [2][TC_A_STAGE_FLOATS]
  float *sB = sA + 2 * TC_A_STAGE_FLOATS;                  // [2][TC_B_STAGE_FLOATS]
  float *s_flux = sB + 2 * TC_B_STAGE_FLOATS;              // [TC_NCOL][TC_FLUX_STRIDE]
  __shared__ __align__(8) uint64_t bars[5];                // fullA[2], empty[2], accfull
  __shared__ uint32_t s_tmem;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t bar_fullA = tc::smem_u32(&bars[0]), bar_empty = tc::smem_u32(&bars[2]), bar_acc = tc::smem_u32(&bars[4]);

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(&s_tmem)), "n"(TC_TMEM_COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid == 32) {
    for (int i = 0; i < 5; ++i) tc::mbar_init(tc::smem_u32(&bars[i]), 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (int i = tid; i < TC_FLUX_FLOATS; i += TC_THREADS) s_flux[i] = 0.f;   // pad columns stay zero
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmain = s_tmem, tsmall = s_tmem + TC_NCOL;
  constexpr uint32_t IDESC = tc::make_idesc(128, TC_NCOL);
  // descriptors of k-step 0 / hi of both stages; every other tile is a multiple of 4 KB (256 x 16 B) further
  const uint64_t descA0 = tc::make_desc(tc::smem_u32(sA), 128 * 16, 128);
  const uint64_t descB0 = tc::make_desc(tc::smem_u32(sB), TC_NCOL * 16, 128);
  constexpr uint32_t TILE16 = TC_TILE_FLOATS * 4 / 16;     // 256

  // this thread's B-production task: column c, node/face-node quad qsub within a k-step
  const int c = warp * 16 + (lane >> 4) * 8 + (lane & 7);
  const int qsub = (lane >> 3) & 1;
  const int ce = c / NF, cf_ = c - ce * NF;                // element within the batch, field

  uint32_t it = 0;        // stages issued so far by this CTA (ring position and mbarrier phases)
  uint32_t bpar = 0;      // accfull parity
  for (int b = blockIdx.x; b < P.nbatch; b += gridDim.x) {
    const int k0 = b * EB;
    const int nvalid = min(EB, p.K - k0);
    const bool cvalid = ce < nvalid && c < EB * NF;

    // ---- per-column pre-combination coefficients (rows a1 + a3): a_j = sum_i cf[j][i] * (u_src[i] - mean)
    float cf[3][3];
    const float *sp[3];
    float mean[3];
    int nsrc = 0;
#pragma unroll
    for (int j = 0; j < 3; ++j)
#pragma unroll
      for (int i = 0; i < 3; ++i) cf[j][i] = 0.f;
    sp[0] = sp[1] = sp[2] = p.q_in;
    mean[0] = mean[1] = mean[2] = 0.f;
    if (cvalid) {
      const float *g = p.geo + (size_t)(k0 + ce) * NGEO;
      float G[9];
#pragma unroll
      for (int i = 0; i < 9; ++i) G[i] = __ldg(g + i);
      int src[3] = {0, 0, 0};
      if (MODEL == 0) {
        const float kap = __ldg(g + 9), irho = __ldg(g + 10);
        if (cf_ == 0) {                 // eq. (5): r_p = -kappa sum_j D_j (sum_i g_ij v_i)
          nsrc = 3;
          src[0] = 1; src[1] = 2; src[2] = 3;
#pragma unroll
          for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int i = 0; i < 3; ++i) cf[j][i] = -kap * G[3 * i + j];
        } else {                        // eq. (6): r_vi = -(1/rho) sum_j g_ij D_j p
          nsrc = 1;
          src[0] = 0;
#pragma unroll
          for (int j = 0; j < 3; ++j) cf[j][0] = -irho * G[3 * (cf_ - 1) + j];
        }
      } else {
        const float irho = __ldg(g + 9), lam = __ldg(g + 10), mu = __ldg(g + 11);
        nsrc = 3;
        if (cf_ < 3) {                  // r_vi = (1/rho) sum_j D_j (sum_m g_mj sigma_im)
          const int row[3][3] = {{3, 6, 7}, {6, 4, 8}, {7, 8, 5}};
#pragma unroll
          for (int m = 0; m < 3; ++m) src[m] = row[cf_][m];
#pragma unroll
          for (int j = 0; j < 3; ++j)
#pragma unroll
            for (int m = 0; m < 3; ++m) cf[j][m] = irho * G[3 * m + j];
        } else {                        // PAPER.md:158 (reading Q6): lambda delta_ab div v + mu (d_b v_a + d_a v_b)
          src[0] = 0; src[1] = 1; src[2] = 2;
          const int a = cf_ < 6 ? cf_ - 3 : (cf_ == 8 ? 1 : 0);
          const int bb = cf_ < 6 ? cf_ - 3 : (cf_ == 6 ? 1 : 2);
#pragma unroll
          for (int j = 0; j < 3; ++j) {
            if (cf_ < 6) {
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
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        sp[i] = p.q_in + ((size_t)(k0 + ce) * NF + src[i]) * NP;
        // mean of the four vertex values: D_j 1 = 0, so the shift is exact and removes the cancellation
        if (i < nsrc) mean[i] = 0.25f * ((__ldg(sp[i]) + __ldg(sp[i] + N)) + (__ldg(sp[i] + NFP - 1) + __ldg(sp[i] + NP - 1)));
      }
    }

    uint32_t acc_main = 0, acc_small = 0;
    for (int st = 0; st < T::NSTAGE; ++st, ++it) {
      const uint32_t s = it & 1, use = it >> 1;
      float *sBs = sB + s * TC_B_STAGE_FLOATS;
      if (it >= 2) tc::mbar_wait(bar_empty + 8 * s, (use - 1) & 1);     // MMAs of the previous use are done
      if (tid == 0) {
        tc::mbar_expect_tx(bar_fullA + 8 * s, TC_A_STAGE_FLOATS * 4);
        tc::bulk_g2s(tc::smem_u32(sA + s * TC_A_STAGE_FLOATS), P.Aimg + (size_t)st * TC_A_STAGE_FLOATS, TC_A_STAGE_FLOATS * 4,
                     bar_fullA + 8 * s);
      }
      if (st < T::NG) {
        // ---- node stage: k-step j = operator D_j applied to nodes 8 st .. 8 st + 7
        const int m0 = 8 * st + 4 * qsub;
        float u[3][4];
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          if (i < nsrc && m0 < NP) {
            if (VEC4) {
              const float4 v = __ldg(reinterpret_cast<const float4 *>(sp[i] + m0));
              u[i][0] = v.x - mean[i]; u[i][1] = v.y - mean[i]; u[i][2] = v.z - mean[i]; u[i][3] = v.w - mean[i];
            } else {
#pragma unroll
              for (int t = 0; t < 4; ++t) u[i][t] = (m0 + t < NP) ? __ldg(sp[i] + m0 + t) - mean[i] : 0.f;
            }
          } else {
            u[i][0] = u[i][1] = u[i][2] = u[i][3] = 0.f;
          }
        }
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          float a[4];
#pragma unroll
          for (int t = 0; t < 4; ++t) a[t] = cf[j][0] * u[0][t] + cf[j][1] * u[1][t] + cf[j][2] * u[2][t];
          float *dst = sBs + j * TC_TILE_FLOATS + qsub * (TC_NCOL * 4) + c * 4;
          tc::split_store(dst, dst + TC_STAGE_K * TC_TILE_FLOATS, a[0], a[1], a[2], a[3]);
        }
      } else {
        // ---- face stage: 24 face nodes; penalty terms into the scratch, then split into the B slice
        const int j0 = (st - T::NG) * 24;
        for (int t = tid; t < EB * 24; t += TC_THREADS) {
          const int e = t / 24, jj = t - e * 24;
          float F[NF];
#pragma unroll
          for (int f = 0; f < NF; ++f) F[f] = 0.f;
          if (e < nvalid && j0 + jj < NFACE) face_node_flux<MODEL, N>(p, k0 + e, j0 + jj, F);
#pragma unroll
          for (int f = 0; f < NF; ++f) s_flux[(e * NF + f) * TC_FLUX_STRIDE + jj] = F[f];
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < TC_STAGE_K; ++r) {
          const float4 v = *reinterpret_cast<const float4 *>(s_flux + c * TC_FLUX_STRIDE + (2 * r + qsub) * 4);
          float *dst = sBs + r * TC_TILE_FLOATS + qsub * (TC_NCOL * 4) + c * 4;
          tc::split_store(dst, dst + TC_STAGE_K * TC_TILE_FLOATS, v.x, v.y, v.z, v.w);
        }
      }
      tc::fence_async_smem();            // generic-proxy writes of B -> visible to the tensor core (async proxy)
      __syncthreads();
      if (tid == 0) {
        tc::mbar_wait(bar_fullA + 8 * s, use & 1);
        tc::tc_fence_after();
        const uint64_t dA = descA0 + (uint64_t)(s * (TC_A_STAGE_FLOATS * 4 / 16));
        const uint64_t dB = descB0 + (uint64_t)(s * (TC_B_STAGE_FLOATS * 4 / 16));
#pragma unroll
        for (int ks = 0; ks < TC_STAGE_K; ++ks) {
          const uint64_t a_hi = dA + (uint64_t)((2 * ks) * TILE16), a_lo = a_hi + TILE16;
          const uint64_t b_hi = dB + (uint64_t)(ks * TILE16), b_lo = b_hi + TC_STAGE_K * TILE16;
          tc::umma_tf32(tsmall, a_lo, b_hi, IDESC, acc_small);
          tc::umma_tf32(tsmall, a_hi, b_lo, IDESC, 1u);
          tc::umma_tf32(tmain, a_hi, b_hi, IDESC, acc_main);
          acc_small = 1u;
          acc_main = 1u;
        }
        tc::umma_commit(bar_empty + 8 * s);
        if (st == T::NSTAGE - 1) tc::umma_commit(bar_acc);
      }
    }

    // ---- epilogue (row a7): thread = node (TMEM lane), 64 columns per warp
    tc::mbar_wait(bar_acc, bpar);
    bpar ^= 1;
    tc::tc_fence_after();
    {
      const int qd = warp & 3, half = warp >> 2;
      const int n = qd * 32 + lane;
      if (qd * 32 < NP) {
#pragma unroll 1
        for (int cb = 0; cb < 2; ++cb) {
          const int c0 = half * 64 + cb * 32;
          if (c0 >= nvalid * NF) break;
          uint32_t vm[32], vs[32];
          tc::tmem_ld32(tmain + ((uint32_t)(qd * 32) << 16) + c0, vm);
          tc::tmem_ld32(tsmall + ((uint32_t)(qd * 32) << 16) + c0, vs);
          if (n < NP) {
            const int ncol = min(32, nvalid * NF - c0);
            const size_t base = ((size_t)k0 * NF + c0) * NP + n;
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              if (j < ncol) {
                const float r = __uint_as_float(vm[j]) + __uint_as_float(vs[j]);
                const size_t idx = base + (size_t)j * NP;
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
          }
        }
      }
    }
    tc::tc_fence_before();
    __syncthreads();          // TMEM drained: the next batch may overwrite the accumulators
  }

  if (warp == 0) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem), "n"(TC_TMEM_COLS) : "memory");
  }
}

}  // namespace dgk
