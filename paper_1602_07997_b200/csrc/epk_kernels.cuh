// Element-per-thread stage kernel of libdg for the lowest degrees (acoustic N = 1, 2; elastic N = 1).
//
// At Np = 4 .. 10 an element's fields fit in one thread's registers (16 .. 40 values), so every row of the hot path
// (a1-a7) runs without shared memory: the fields and the residual move as 16-byte vectors, the
// reference operators D_r, D_s, D_t and LIFT sit in constant memory and enter the FFMAs as constant-bank operands (all
// loops are fully unrolled, every register index is a compile-time constant), and the only irregular access is the gather
// of the exterior traces through the compressed connectivity.  The generic fused SIMT kernel (kernels.cuh) is bound by
// its shared-memory operand traffic at these degrees (L1/LSU pipe 98 % busy at N = 1).
//
// Prior art: the one-element-per-thread kernels of PAPER.md:173 (K1-K3, element-fastest layout, operators prefetched to
// shared memory); here the node-fastest ABI layout is kept (an element is one contiguous run), the three kernels are
// fused with the LSRK update, and the operators need no staging.  The arithmetic (vertex-mean shift, pre-/post-
// combination order, penalty terms) is the one of kernels.cuh.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "flux.cuh"
#include "kernels.cuh"

// (development switches of the warp-cooperative staging paths below; the defaults are the measured best)
#ifndef DG_X_EPK_GIN
#define DG_X_EPK_GIN 1
#endif
#ifndef DG_X_EPK_QIN
#define DG_X_EPK_QIN 0
#endif
#ifndef DG_X_EPK_GINE
#define DG_X_EPK_GINE 1      // elastic N = 1: records through the tile
#endif
#ifndef DG_X_EPK_F2
#define DG_X_EPK_F2 1          // volume and lift FMAs as FFMA2 on node pairs
#endif
#ifndef DG_X_EPK_COUT
#define DG_X_EPK_COUT 1
#endif
#ifndef DG_X_EPK_VGE
#define DG_X_EPK_VGE 1
#endif
#ifndef DG_X_EPK_COUTE
#define DG_X_EPK_COUTE 1     // elastic N = 1: results through the tile
#endif
#ifndef DG_X_EPK_QINE
#define DG_X_EPK_QINE 0      // elastic N = 1 fields through the tile: 1.27 -> 1.32 ms: off
#endif

namespace dgk {

constexpr int EPK_MAXNP = 10, EPK_MAXNFP = 6, EPK_MAXNFACE = 24;     // N <= 2
static __constant__ float c_epk_D[3 * EPK_MAXNP * EPK_MAXNP];          // D_j[n][m] at (j Np + n) Np + m
static __constant__ float c_epk_L[EPK_MAXNP * EPK_MAXNFACE];           // LIFT[n][j] at n 4Nfp + j
// the same operators with the output node n fastest, so that a pair (n, n + 1) is one 64-bit constant-bank operand of FFMA2
static __constant__ float c_epk_Dt[3 * EPK_MAXNP * EPK_MAXNP];         // D_j[n][m] at (j Np + m) Np + n
static __constant__ float c_epk_Lt[EPK_MAXNFACE * EPK_MAXNP];          // LIFT[n][j] at j Np + n
static __constant__ unsigned short c_epk_nbrnode[4 * 24 * EPK_MAXNFP]; // neighbour's volume node at (f 24 + code) Nfp + i

// face masks in the library's order (host_setup.cpp: nodes in lattice order, t slowest, r fastest; a face lists its
// nodes by increasing number) as compile-time constants, so that interior traces are register reads
template <int N>
struct EpkFmask {
  static constexpr int NFP = (N + 1) * (N + 2) / 2;
  int v[4 * NFP];
  constexpr EpkFmask() : v{} {
    int cnt[4] = {0, 0, 0, 0};
    int n = 0;
    for (int k = 0; k <= N; ++k)
      for (int j = 0; j <= N - k; ++j)
        for (int i = 0; i <= N - k - j; ++i, ++n) {
          if (k == 0) v[0 * NFP + cnt[0]++] = n;             // t = -1
          if (j == 0) v[1 * NFP + cnt[1]++] = n;             // s = -1
          if (i + j + k == N) v[2 * NFP + cnt[2]++] = n;     // r + s + t = -1
          if (i == 0) v[3 * NFP + cnt[3]++] = n;             // r = -1
        }
  }
};

// resident CTAs per SM asked of the compiler: the kernel is bound by the latency of its scattered gathers, so occupancy pays
// as long as the register cap does not spill much (same-box A/B, ms per stage: acoustic N = 1 0.752 -> 0.713 with six CTAs;
// elastic N = 1 1.772 -> 1.658 and acoustic N = 2 0.801 -> 0.789 with four; five or six CTAs there spill and lose 12-75 %).
// With the records staged through shared memory (below) acoustic N = 1 is best at five: 0.603 (six, spills) -> 0.556.
// Elastic N = 1 with whole-vector trace gathers (36 more live registers) wants three: 2.00 (four, 700 bytes of spills) -> 1.51;
// with records and results through the tiles on top 1.27 (two CTAs 1.45, four 2.14).
template <int MODEL, int N>
constexpr int epk_min_ctas() {
#ifdef DG_X_EPK_MINB
  return DG_X_EPK_MINB;
#else
  return N == 1 ? (MODEL == 0 ? 5 : 3) : 4;
#endif
}

template <int MODEL, int N, int MODE>
__global__ void __launch_bounds__(128, epk_min_ctas<MODEL, N>()) epk_stage_kernel(const StageParams p) {
  using D = Deg<N>;
  constexpr int NP = D::NP, NFP = D::NFP, NFACE = D::NFACE;
  constexpr int NF = MODEL == 0 ? 4 : 9, NGEO = MODEL == 0 ? GEO_AC : GEO_EL;
  constexpr int NV = NF * NP;                                          // values per element
  static_assert(NV % 4 == 0, "an element's fields are moved as 16-byte vectors");
  constexpr EpkFmask<N> FM{};
  constexpr bool F2 = DG_X_EPK_F2 && NP == 4;                          // (N = 2: the pairs cost registers the kernel does not have: 356 bytes of spills)
  // N = 1, acoustic: an element is four 16-byte vectors (one per field), and the four lanes of a quad gather their
  // neighbours' elements together (below): every lane stays alive, lanes beyond the range redo the last element and store nothing
  constexpr bool COOP = NP == 4 && MODEL == 0;
  constexpr bool EL1 = MODEL == 1 && NP == 4;                          // elastic N = 1: nine vectors per element
  constexpr int XP = (NV / 4) | 1;                                     // row pitch of the tile in vectors: odd (conflict-free)
  __shared__ float4 s_x[(COOP || (EL1 && (DG_X_EPK_COUTE || DG_X_EPK_QINE))) ? 128 * XP : 1];   // per thread a padded row
  const int k_raw = p.kbeg + blockIdx.x * blockDim.x + threadIdx.x;
  constexpr bool ALIVE = COOP || (MODEL == 1 && NP == 4 && (DG_X_EPK_GINE || DG_X_EPK_COUTE || DG_X_EPK_QINE));   // warp-cooperative staging: every lane stays
  if (!ALIVE && k_raw >= p.K) return;
  const bool active = k_raw < p.K;
  const int k = active ? k_raw : p.K - 1;

  // ---- per-element constants and fields
  // the element's record: G[9], materials, 4 face records -- whole in registers for the acoustic model (32 values),
  // the first 16 for the elastic one (its face records are read through L1 when needed: register pressure)
  constexpr int NGL = MODEL == 0 ? NGEO : 16;
  const float *g = p.geo + (size_t)k * NGEO;
  // N = 1, acoustic: the warp's 32 geometric records (4 KB) and field rows (2 KB) are contiguous runs: the warp loads them
  // four lines per instruction into padded shared-memory rows and every lane picks up its own (a 16-byte load per lane at
  // a stride of 128 | 64 bytes touches 32 | 16 lines per instruction; the kernel is bound by exactly those L1 tag lookups)
  constexpr bool GIN = (COOP && DG_X_EPK_GIN) || (MODEL == 1 && NP == 4 && DG_X_EPK_GINE), QIN = (COOP && DG_X_EPK_QIN) || (EL1 && DG_X_EPK_QINE);
  constexpr int GP4 = NGEO / 4 + 1;                                    // row pitch of the record tile, in vectors: odd
  __shared__ float4 s_g[GIN ? 128 * GP4 : 1];
  const int lane_ = threadIdx.x & 31, kw_ = k_raw - lane_, nvalid_ = min(32, p.K - kw_);
  if (nvalid_ <= 0) return;                                            // (a warp wholly beyond the range)
  float gl[NGL];
  if (GIN) {
    float4 *gwarp = s_g + (threadIdx.x & ~31) * GP4;
    const float4 *gsrc = reinterpret_cast<const float4 *>(p.geo) + (size_t)kw_ * (NGEO / 4);
#pragma unroll
    for (int it = 0; it < NGEO / 4; ++it) {
      const int idx = it * 32 + lane_, e = idx / (NGEO / 4), v = idx - e * (NGEO / 4);
      gwarp[e * GP4 + v] = __ldg(gsrc + (size_t)min(e, nvalid_ - 1) * (NGEO / 4) + v);
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < NGL / 4; ++i) {
      const float4 v = s_g[threadIdx.x * GP4 + i];
      gl[4 * i] = v.x; gl[4 * i + 1] = v.y; gl[4 * i + 2] = v.z; gl[4 * i + 3] = v.w;
    }
  } else {
#pragma unroll
    for (int i = 0; i < NGL / 4; ++i) {
      const float4 v = __ldg(reinterpret_cast<const float4 *>(g) + i);
      gl[4 * i] = v.x; gl[4 * i + 1] = v.y; gl[4 * i + 2] = v.z; gl[4 * i + 3] = v.w;
    }
  }
  float q[NV], r[NV];
  if (QIN) {
    float4 *xwarp = s_x + (threadIdx.x & ~31) * XP;
    const float4 *qsrc = reinterpret_cast<const float4 *>(p.q_in) + (size_t)kw_ * (NV / 4);
#pragma unroll
    for (int it = 0; it < NV / 4; ++it) {
      const int idx = it * 32 + lane_, e = idx / (NV / 4), v = idx - e * (NV / 4);
      xwarp[e * XP + v] = __ldg(qsrc + (size_t)min(e, nvalid_ - 1) * (NV / 4) + v);
    }
    __syncwarp();
#pragma unroll
    for (int i = 0; i < NV / 4; ++i) {
      const float4 v = s_x[threadIdx.x * XP + i];
      q[4 * i] = v.x; q[4 * i + 1] = v.y; q[4 * i + 2] = v.z; q[4 * i + 3] = v.w;
    }
    __syncwarp();                                                      // (the rows are reused by the face gather)
  } else {
    const float4 *src = reinterpret_cast<const float4 *>(p.q_in + (size_t)k * NV);
#pragma unroll
    for (int i = 0; i < NV / 4; ++i) {
      const float4 v = __ldg(src + i);
      q[4 * i] = v.x; q[4 * i + 1] = v.y; q[4 * i + 2] = v.z; q[4 * i + 3] = v.w;
    }
  }

  // ---- volume term (rows a1-a3).  Inputs of a differentiation are shifted by the mean of the four vertex values
  // (D_j 1 = 0)
  float u[NV];
#pragma unroll
  for (int f = 0; f < NF; ++f) {
    const float mean = 0.25f * ((q[f * NP] + q[f * NP + N]) + (q[f * NP + NFP - 1] + q[f * NP + NP - 1]));
#pragma unroll
    for (int m = 0; m < NP; ++m) u[f * NP + m] = q[f * NP + m] - mean;
  }
  if (MODEL == 0) {
    // eq. (5): w_j = sum_i g_ij v_i
    float w[3][NP];
#pragma unroll
    for (int m = 0; m < NP; ++m) {
      w[0][m] = gl[0] * u[NP + m] + gl[3] * u[2 * NP + m] + gl[6] * u[3 * NP + m];
      w[1][m] = gl[1] * u[NP + m] + gl[4] * u[2 * NP + m] + gl[7] * u[3 * NP + m];
      w[2][m] = gl[2] * u[NP + m] + gl[5] * u[2 * NP + m] + gl[8] * u[3 * NP + m];
    }
    const float kap = gl[9], irho = gl[10];
#pragma unroll
    for (int n = 0; n < NP; n += 2) {
      // two output nodes per FFMA2 (the packed FP32 FMA of sm_100): the operator pair (n, n + 1) is one 64-bit constant operand
      float2 A0 = make_float2(0.f, 0.f), A1 = A0, A2 = A0, A3 = A0;
      float a0[2] = {0.f, 0.f}, a1[2] = {0.f, 0.f}, a2[2] = {0.f, 0.f}, a3[2] = {0.f, 0.f};
#pragma unroll
      for (int m = 0; m < NP; ++m) {
        if (F2) {
          const float2 DR = make_float2(c_epk_Dt[(0 * NP + m) * NP + n], c_epk_Dt[(0 * NP + m) * NP + n + 1]);
          const float2 DS = make_float2(c_epk_Dt[(1 * NP + m) * NP + n], c_epk_Dt[(1 * NP + m) * NP + n + 1]);
          const float2 DT = make_float2(c_epk_Dt[(2 * NP + m) * NP + n], c_epk_Dt[(2 * NP + m) * NP + n + 1]);
          const float2 um = make_float2(u[m], u[m]);
          A0 = __ffma2_rn(DR, um, A0);
          A1 = __ffma2_rn(DS, um, A1);
          A2 = __ffma2_rn(DT, um, A2);
          A3 = __ffma2_rn(DR, make_float2(w[0][m], w[0][m]), A3);
          A3 = __ffma2_rn(DS, make_float2(w[1][m], w[1][m]), A3);
          A3 = __ffma2_rn(DT, make_float2(w[2][m], w[2][m]), A3);
        } else {
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const float dr = c_epk_D[(0 * NP + n + h) * NP + m], ds = c_epk_D[(1 * NP + n + h) * NP + m], dt = c_epk_D[(2 * NP + n + h) * NP + m];
            a0[h] = fmaf(dr, u[m], a0[h]);
            a1[h] = fmaf(ds, u[m], a1[h]);
            a2[h] = fmaf(dt, u[m], a2[h]);
            a3[h] = fmaf(dr, w[0][m], a3[h]);
            a3[h] = fmaf(ds, w[1][m], a3[h]);
            a3[h] = fmaf(dt, w[2][m], a3[h]);
          }
        }
      }
      if (F2) {
        a0[0] = A0.x; a0[1] = A0.y; a1[0] = A1.x; a1[1] = A1.y; a2[0] = A2.x; a2[1] = A2.y; a3[0] = A3.x; a3[1] = A3.y;
      }
      // eq. (5)-(6)
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        r[n + h] = -kap * a3[h];
#pragma unroll
        for (int i = 0; i < 3; ++i) r[(1 + i) * NP + n + h] = -irho * (gl[3 * i] * a0[h] + gl[3 * i + 1] * a1[h] + gl[3 * i + 2] * a2[h]);
      }
    }
  } else {
    // w_{i,n} = sum_m g_mn sigma_im ; fields vx vy vz sxx syy szz sxy sxz syz
    const float irho = gl[9], lam = gl[10], mu = gl[11];
    constexpr int SG[3][3] = {{3, 6, 7}, {6, 4, 8}, {7, 8, 5}};
    float w[3][3][NP];                                                 // w[i][j][m] = sum_c g_cj sigma_ic
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
      for (int m = 0; m < NP; ++m) {
        const float s0 = u[SG[i][0] * NP + m], s1 = u[SG[i][1] * NP + m], s2 = u[SG[i][2] * NP + m];
        w[i][0][m] = gl[0] * s0 + gl[3] * s1 + gl[6] * s2;
        w[i][1][m] = gl[1] * s0 + gl[4] * s1 + gl[7] * s2;
        w[i][2][m] = gl[2] * s0 + gl[5] * s1 + gl[8] * s2;
      }
#pragma unroll
    for (int n2 = 0; n2 < NP; n2 += 2) {
      float2 ACC[12];
#pragma unroll
      for (int c = 0; c < 12; ++c) ACC[c] = make_float2(0.f, 0.f);
      float accs[2][12];
#pragma unroll
      for (int c = 0; c < 12; ++c) accs[0][c] = accs[1][c] = 0.f;
#pragma unroll
      for (int m = 0; m < NP; ++m) {
        if (F2) {
          const float2 DR = make_float2(c_epk_Dt[(0 * NP + m) * NP + n2], c_epk_Dt[(0 * NP + m) * NP + n2 + 1]);
          const float2 DS = make_float2(c_epk_Dt[(1 * NP + m) * NP + n2], c_epk_Dt[(1 * NP + m) * NP + n2 + 1]);
          const float2 DT = make_float2(c_epk_Dt[(2 * NP + m) * NP + n2], c_epk_Dt[(2 * NP + m) * NP + n2 + 1]);
#pragma unroll
          for (int i = 0; i < 3; ++i) {
            const float2 ui = make_float2(u[i * NP + m], u[i * NP + m]);
            ACC[3 * i + 0] = __ffma2_rn(DR, ui, ACC[3 * i + 0]);
            ACC[3 * i + 1] = __ffma2_rn(DS, ui, ACC[3 * i + 1]);
            ACC[3 * i + 2] = __ffma2_rn(DT, ui, ACC[3 * i + 2]);
            ACC[9 + i] = __ffma2_rn(DR, make_float2(w[i][0][m], w[i][0][m]), ACC[9 + i]);
            ACC[9 + i] = __ffma2_rn(DS, make_float2(w[i][1][m], w[i][1][m]), ACC[9 + i]);
            ACC[9 + i] = __ffma2_rn(DT, make_float2(w[i][2][m], w[i][2][m]), ACC[9 + i]);
          }
        } else {
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const float dr = c_epk_D[(0 * NP + n2 + h) * NP + m], ds = c_epk_D[(1 * NP + n2 + h) * NP + m], dt = c_epk_D[(2 * NP + n2 + h) * NP + m];
#pragma unroll
            for (int i = 0; i < 3; ++i) {
              accs[h][3 * i + 0] = fmaf(dr, u[i * NP + m], accs[h][3 * i + 0]);
              accs[h][3 * i + 1] = fmaf(ds, u[i * NP + m], accs[h][3 * i + 1]);
              accs[h][3 * i + 2] = fmaf(dt, u[i * NP + m], accs[h][3 * i + 2]);
              accs[h][9 + i] = fmaf(dr, w[i][0][m], accs[h][9 + i]);
              accs[h][9 + i] = fmaf(ds, w[i][1][m], accs[h][9 + i]);
              accs[h][9 + i] = fmaf(dt, w[i][2][m], accs[h][9 + i]);
            }
          }
        }
      }
#pragma unroll
      for (int h = 0; h < 2; ++h) {
      const int n = n2 + h;
      float acc[12];
#pragma unroll
      for (int c = 0; c < 12; ++c) acc[c] = F2 ? (h == 0 ? ACC[c].x : ACC[c].y) : accs[h][c];
      float gv[3][3];   // gv[i][j] = d_j v_i = sum_m g_jm (D_m v_i)
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) gv[i][j] = gl[3 * j] * acc[3 * i] + gl[3 * j + 1] * acc[3 * i + 1] + gl[3 * j + 2] * acc[3 * i + 2];
      const float div = gv[0][0] + gv[1][1] + gv[2][2];
      r[0 * NP + n] = irho * acc[9];
      r[1 * NP + n] = irho * acc[10];
      r[2 * NP + n] = irho * acc[11];
      r[3 * NP + n] = lam * div + 2.f * mu * gv[0][0];
      r[4 * NP + n] = lam * div + 2.f * mu * gv[1][1];
      r[5 * NP + n] = lam * div + 2.f * mu * gv[2][2];
      r[6 * NP + n] = mu * (gv[0][1] + gv[1][0]);
      r[7 * NP + n] = mu * (gv[0][2] + gv[2][0]);
      r[8 * NP + n] = mu * (gv[1][2] + gv[2][1]);
      }
    }
  }

  // ---- surface term (rows a4-a6): gather, penalty terms times g^sur, lift
  // the element's connectivity as two vector loads (the kernel is bound by its load / store instructions, not by DRAM)
  const int4 nbr4 = __ldg(reinterpret_cast<const int4 *>(p.nbr) + k);
  const unsigned code4 = __ldg(reinterpret_cast<const unsigned *>(p.fcode) + k);
#pragma unroll
  for (int f = 0; f < 4; ++f) {
    constexpr int FO = MODEL == 0 ? 12 : 16, FS = MODEL == 0 ? 5 : 8;
    float fg[8];
    if (MODEL == 1 && GIN) {                                             // elastic: the face record from this thread's row of the tile
      const float4 a = s_g[threadIdx.x * GP4 + (GIN ? (FO + FS * f) / 4 : 0)], b = s_g[threadIdx.x * GP4 + (GIN ? (FO + FS * f) / 4 + 1 : 0)];
      fg[0] = a.x; fg[1] = a.y; fg[2] = a.z; fg[3] = a.w; fg[4] = b.x; fg[5] = b.y; fg[6] = b.z; fg[7] = b.w;
    } else {
#pragma unroll
      for (int i = 0; i < FS; ++i) fg[i] = MODEL == 0 ? gl[(FO + FS * f + i) % NGL] : __ldg(g + FO + FS * f + i);
    }
    const float nx = fg[0], ny = fg[1], nz = fg[2];
    const int nb = f == 0 ? nbr4.x : (f == 1 ? nbr4.y : (f == 2 ? nbr4.z : nbr4.w));      // (f is a compile-time constant: unrolled)
    const int code = (int)((code4 >> (8 * f)) & 255u);
    // N = 1: a field of the neighbour is one 16-byte vector (Np = 4): fetch it whole and pick the node afterwards
    // (a third of the gather instructions; the kernel is bound by the L1/LSU pipe, the ALUs are idle)
    // (elastic: nine vectors per face, this lane's own neighbour: a third of the load instructions and of the L1 wavefronts --
    // ncu had 9 wavefronts per scalar gather request; same-box A/B 1.62 -> 1.51 ms per stage, dg_rhs 1.33 -> 1.09, at three CTAs per SM)
    constexpr bool VGATHER = COOP || (MODEL == 1 && NP == 4 && DG_X_EPK_VGE);
    float4 nq[VGATHER ? NF : 1];
    if (VGATHER && !COOP && !p.pflux) {                                  // elastic N = 1: this lane's neighbour, nine whole vectors
      if (nb >= 0) {
#pragma unroll
        for (int c = 0; c < NF; ++c) nq[c] = __ldg(reinterpret_cast<const float4 *>(p.q_in + (size_t)nb * NV) + c);
      }
    }
    if (COOP && !p.pflux) {
      // Warp-level gather: the kernel is bound by the L1 tag stage (one 128-byte line per lane and load: 32 lines per warp
      // instruction).  Lane j of a quad loads vector j (= field j) of the neighbour of each of the quad's four elements in
      // turn -- 8 lines per warp instruction instead of 32 -- and the quad transposes the 4 x 4 vectors through a padded
      // shared-memory row per lane (conflict-free 16-byte accesses).
      const int lane = threadIdx.x & 31, qj = lane & 3, qb = lane & ~3;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int nbi = __shfl_sync(0xffffffffu, nb, qb + i);
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (nbi >= 0) v = __ldg(reinterpret_cast<const float4 *>(p.q_in + (size_t)nbi * NV) + qj);
        s_x[((threadIdx.x & ~3) + i) * XP + qj] = v;
      }
      __syncwarp();
#pragma unroll
      for (int c = 0; c < NF; ++c) nq[c] = s_x[threadIdx.x * XP + c];
      __syncwarp();
    }
    auto pick = [](const float4 &v, int nn) { return (nn & 2) ? ((nn & 1) ? v.w : v.z) : ((nn & 1) ? v.y : v.x); };
#pragma unroll
    for (int i = 0; i < NFP; ++i) {
      const int j = f * NFP + i;
      const int nm = FM.v[f * NFP + i];                                // compile-time: q[] stays in registers
      float um[NF], F[NF];
#pragma unroll
      for (int c = 0; c < NF; ++c) um[c] = q[c * NP + nm];
      if (p.pflux) {                                                   // interface-centric surface step: terms from the face buffer
#pragma unroll
        for (int c = 0; c < NF; ++c) F[c] = __ldg(p.pflux + ((size_t)k * NF + c) * NFACE + j);
      } else if (MODEL == 0) {
        float dp, dvn;
        if (nb >= 0) {
          const int nn = c_epk_nbrnode[(f * 24 + code) * NFP + i];
          float up[4];
          if (VGATHER) {
#pragma unroll
            for (int c = 0; c < 4; ++c) up[c] = pick(nq[c], nn);
          } else {
            const float *qp = p.q_in + (size_t)nb * NV + nn;
#pragma unroll
            for (int c = 0; c < 4; ++c) up[c] = __ldg(qp + c * NP);
          }
          dp = up[0] - um[0];
          dvn = (up[1] - um[1]) * nx + (up[2] - um[2]) * ny + (up[3] - um[3]) * nz;
        } else {
          acoustic_boundary_jump(nb, um[0], um[1] * nx + um[2] * ny + um[3] * nz, dp, dvn);
        }
        const float4 Pn = acoustic_penalty(gl, fg, dp, dvn);
        F[0] = Pn.x; F[1] = Pn.y; F[2] = Pn.z; F[3] = Pn.w;
      } else {
        float Tmx, Tmy, Tmz;
        traction(um, nx, ny, nz, Tmx, Tmy, Tmz);
        float dv[3], dT[3];
        if (nb >= 0) {
          const int nn = c_epk_nbrnode[(f * 24 + code) * NFP + i];
          float up[NF];
          if (VGATHER) {
#pragma unroll
            for (int c = 0; c < NF; ++c) up[c] = pick(nq[c], nn);
          } else {
            const float *qp = p.q_in + (size_t)nb * NV + nn;
#pragma unroll
            for (int c = 0; c < NF; ++c) up[c] = __ldg(qp + c * NP);
          }
          float Tpx, Tpy, Tpz;
          traction(up, nx, ny, nz, Tpx, Tpy, Tpz);
          dv[0] = up[0] - um[0]; dv[1] = up[1] - um[1]; dv[2] = up[2] - um[2];
          dT[0] = Tpx - Tmx; dT[1] = Tpy - Tmy; dT[2] = Tpz - Tmz;
        } else {
          elastic_boundary_jump(nb, um, Tmx, Tmy, Tmz, nx, ny, nz, dv, dT);
        }
        elastic_penalty(gl, fg, dv, dT, F);
      }
      if (F2) {
#pragma unroll
        for (int n = 0; n < NP; n += 2) {
          const float2 l2 = make_float2(c_epk_Lt[j * NP + n], c_epk_Lt[j * NP + n + 1]);
#pragma unroll
          for (int c = 0; c < NF; ++c) {
            const float2 rp = __ffma2_rn(l2, make_float2(F[c], F[c]), make_float2(r[c * NP + n], r[c * NP + n + 1]));
            r[c * NP + n] = rp.x;
            r[c * NP + n + 1] = rp.y;
          }
        }
      } else {
#pragma unroll
        for (int n = 0; n < NP; ++n) {
          const float l = c_epk_L[n * NFACE + j];
#pragma unroll
          for (int c = 0; c < NF; ++c) r[c * NP + n] = fmaf(l, F[c], r[c * NP + n]);
        }
      }
    }
  }

  // ---- LSRK update (row a7), 16-byte vectors
  if ((COOP && DG_X_EPK_COUT) || (EL1 && DG_X_EPK_COUTE)) {
    // N = 1, acoustic: a thread's element is a 64-byte run, so a vector store per lane touches 16 lines per warp instruction.
    // Results leave through the padded shared-memory rows instead, and the warp writes its 32 elements -- one contiguous
    // 2 KB run -- four lines per instruction.
    const int lane = threadIdx.x & 31;
    const int kw = k_raw - lane, nvalid = min(32, p.K - kw);
    float4 *srow = s_x + threadIdx.x * XP, *swarp = s_x + (threadIdx.x & ~31) * XP;
    auto put = [&](const float *x) {
#pragma unroll
      for (int i = 0; i < NV / 4; ++i) srow[i] = make_float4(x[4 * i], x[4 * i + 1], x[4 * i + 2], x[4 * i + 3]);
    };
    auto out = [&](float *gdst) {
      __syncwarp();
      float4 *dst = reinterpret_cast<float4 *>(gdst + (size_t)kw * NV);
#pragma unroll
      for (int it = 0; it < NV / 4; ++it) {
        const int idx = it * 32 + lane, e = idx / (NV / 4), v = idx - e * (NV / 4);
        if (e < nvalid) dst[idx] = swarp[e * XP + v];
      }
      __syncwarp();
    };
    const size_t base = (size_t)k * NV;
    if (MODE == MODE_RHS) {
      put(r);
      out(p.rhs);
    } else if (MODE == MODE_AB3) {
      const float4 *h1 = reinterpret_cast<const float4 *>(p.res + base), *h2 = reinterpret_cast<const float4 *>(p.hist2 + base);
#pragma unroll
      for (int i = 0; i < NV / 4; ++i) {
        const float4 x = h1[i], y = __ldg(h2 + i);
        q[4 * i] = fmaf(p.b, y.x, fmaf(p.a, x.x, fmaf(p.dt, r[4 * i], q[4 * i])));
        q[4 * i + 1] = fmaf(p.b, y.y, fmaf(p.a, x.y, fmaf(p.dt, r[4 * i + 1], q[4 * i + 1])));
        q[4 * i + 2] = fmaf(p.b, y.z, fmaf(p.a, x.z, fmaf(p.dt, r[4 * i + 2], q[4 * i + 2])));
        q[4 * i + 3] = fmaf(p.b, y.w, fmaf(p.a, x.w, fmaf(p.dt, r[4 * i + 3], q[4 * i + 3])));
      }
      __syncwarp();                                                    // (every lane has read its history rows: p.rhs may alias none of them, but keep order)
      put(r);
      out(p.rhs);
      put(q);
      out(p.q_out);
    } else {
      const float4 *pres = reinterpret_cast<const float4 *>(p.res + base);
#pragma unroll
      for (int i = 0; i < NV / 4; ++i) {
        float rs[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) rs[t] = p.dt * r[4 * i + t];
        if (p.a != 0.f) {
          const float4 o = pres[i];
          rs[0] = fmaf(p.a, o.x, rs[0]); rs[1] = fmaf(p.a, o.y, rs[1]); rs[2] = fmaf(p.a, o.z, rs[2]); rs[3] = fmaf(p.a, o.w, rs[3]);
        }
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          r[4 * i + t] = rs[t];
          q[4 * i + t] = fmaf(p.b, rs[t], q[4 * i + t]);
        }
      }
      put(r);
      out(p.res);
      put(q);
      out(p.q_out);
    }
    return;
  }
  if (!active) return;                                                 // (lanes kept alive for the quad gather only)
  const size_t base = (size_t)k * NV;
  if (MODE == MODE_RHS) {
    float4 *dst = reinterpret_cast<float4 *>(p.rhs + base);
#pragma unroll
    for (int i = 0; i < NV / 4; ++i) dst[i] = make_float4(r[4 * i], r[4 * i + 1], r[4 * i + 2], r[4 * i + 3]);
  } else if (MODE == MODE_AB3) {
    float4 *dst = reinterpret_cast<float4 *>(p.rhs + base), *pq = reinterpret_cast<float4 *>(p.q_out + base);
    const float4 *h1 = reinterpret_cast<const float4 *>(p.res + base), *h2 = reinterpret_cast<const float4 *>(p.hist2 + base);
#pragma unroll
    for (int i = 0; i < NV / 4; ++i) {
      const float4 x = h1[i], y = __ldg(h2 + i);
      dst[i] = make_float4(r[4 * i], r[4 * i + 1], r[4 * i + 2], r[4 * i + 3]);
      pq[i] = make_float4(fmaf(p.b, y.x, fmaf(p.a, x.x, fmaf(p.dt, r[4 * i], q[4 * i]))),
                          fmaf(p.b, y.y, fmaf(p.a, x.y, fmaf(p.dt, r[4 * i + 1], q[4 * i + 1]))),
                          fmaf(p.b, y.z, fmaf(p.a, x.z, fmaf(p.dt, r[4 * i + 2], q[4 * i + 2]))),
                          fmaf(p.b, y.w, fmaf(p.a, x.w, fmaf(p.dt, r[4 * i + 3], q[4 * i + 3]))));
    }
  } else {
    float4 *pres = reinterpret_cast<float4 *>(p.res + base), *pq = reinterpret_cast<float4 *>(p.q_out + base);
#pragma unroll
    for (int i = 0; i < NV / 4; ++i) {
      float rs[4];
#pragma unroll
      for (int t = 0; t < 4; ++t) rs[t] = p.dt * r[4 * i + t];
      if (p.a != 0.f) {
        const float4 o = pres[i];
        rs[0] = fmaf(p.a, o.x, rs[0]); rs[1] = fmaf(p.a, o.y, rs[1]); rs[2] = fmaf(p.a, o.z, rs[2]); rs[3] = fmaf(p.a, o.w, rs[3]);
      }
      pres[i] = make_float4(rs[0], rs[1], rs[2], rs[3]);
      pq[i] = make_float4(fmaf(p.b, rs[0], q[4 * i]), fmaf(p.b, rs[1], q[4 * i + 1]), fmaf(p.b, rs[2], q[4 * i + 2]),
                          fmaf(p.b, rs[3], q[4 * i + 3]));
    }
  }
}

}  // namespace dgk
