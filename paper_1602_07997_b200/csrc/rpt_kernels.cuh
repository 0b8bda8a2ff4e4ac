// Row-per-thread stage kernel of libdg for the low degrees (N = 1 .. 3), variant 5: "simt_row_per_thread".
//
// A thread owns one row (element, field) of the state: its Np right-hand-side values live in registers, and the whole
// path (rows a1-a7) runs as FP32 FMAs whose operator operand comes from the constant bank
//
//     r[n] += D_j[n][m] * a_j[m]      a_j[m] = sum_i cf[j][i] (u_src_i[m] - mean_i)      (rows a1-a3; eq. (5)-(6))
//     r[n] += LIFT[n][j] * F[j]                                                          (row a6)
//
// with m (resp. the face node j) in the outer, fully unrolled loop, so that every FFMA reads its D / LIFT entry as an
// immediate constant-bank operand, consecutive FFMAs walk consecutive constant addresses, and no operator value passes
// through the load/store pipe (the generic fused kernel, kernels.cuh, is bound by exactly that traffic at these degrees;
// the tensor-core kernel spends three of four k-steps on padding at N = 2 and pays its BF16x3 split per value).
// The lanes of a warp are the Nf rows of 8 (acoustic) / 3 (elastic; 27 of 32 lanes) consecutive elements: a tile.  Warps are
// persistent and work alone (no CTA-wide barrier): each walks over tiles with two shared-memory slots, the next tile's
// fields, geometric records and connectivity landing through cp.async (4 bytes each: odd row pitches keep the scalar reads
// conflict-free) while the current one is worked on; pre-combination sources, interior traces and the own row are read
// from the slot.  The 4 Nfp face nodes of an element are shared out over its Nf lanes (a4, a5:
// gather through the compressed connectivity, penalty terms of flux.cuh), pass through a second tile, and each lane lifts
// its own field.  The arithmetic (vertex-mean shift, row coefficients, penalty terms) is the one of the other two families.
//
// Prior art: the one-node-per-thread kernels of PAPER.md:175 (operators in shared memory); the thread = (element, field)
// mapping with constant-bank operators is this library's.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "flux.cuh"
#include "kernels.cuh"
#include "tc3_kernels.cuh"   // row_coefficients_s

namespace dgk {

constexpr int RPT_MAXN = 3, RPT_MAXNP = 20, RPT_MAXNFACE = 40;
#if !defined(DG_N) || DG_N <= 3
static __constant__ float c_rpt_D[3 * RPT_MAXNP * RPT_MAXNP];   // D_j[n][m] at (3 m + j) Np + n
static __constant__ float c_rpt_L[RPT_MAXNFACE * RPT_MAXNP];    // LIFT[n][j] at j Np + n
#else
static __constant__ float c_rpt_D[1], c_rpt_L[1];
#endif

template <int MODEL, int N>
struct Rpt {
  using D = Deg<N>;
  static constexpr int NP = D::NP, NFP = D::NFP, NFACE = D::NFACE;
  static constexpr int NF = MODEL == 0 ? 4 : 9, NGEO = MODEL == 0 ? GEO_AC : GEO_EL;
  static constexpr int EPW = 32 / NF;                      // elements per warp
  static constexpr int ROWS = EPW * NF;                    // active lanes
  static constexpr int NPP = NP | 1;                       // tile row pitch (floats): odd, scalar reads conflict-free
  // penalty-term row pitch (floats): = 1 mod 8 (acoustic) / mod 32 (elastic), so that with face node j = f + Nf t on
  // lane (el, f) the stores of a warp (bank = Nf el + f + const) and the row reads of the lift are conflict-free
  static constexpr int FQ = MODEL == 0 ? 8 : 32, FP = (NFACE + FQ - 2) / FQ * FQ + 1;
  static constexpr int TPL = (NFACE + NF - 1) / NF;        // face nodes per lane
  static constexpr int VW = NP % 4 == 0 ? 4 : (NP % 2 == 0 ? 2 : 1);   // vector width of row accesses (floats)
  static constexpr int GP = NGEO | 1;                      // pitch of a geometric record in the tile: odd
  static constexpr int WARPS = N <= 2 ? 2 : 1;                          // warps per CTA (each warp works alone; static shared memory < 48 KB)
  static constexpr int EPC = WARPS * EPW;                  // elements per CTA
};

template <int VW>
struct RptVec;
template <>
struct RptVec<4> { using T = float4; };
template <>
struct RptVec<2> { using T = float2; };
template <>
struct RptVec<1> { using T = float; };

// resident CTAs per SM asked of the compiler (same-box A/B, ms per stage, persistent version: N = 2 eight CTAs of two warps
// and 128 registers -- acoustic 0.743, elastic 1.98; N = 3 twelve CTAs of one warp -- acoustic 1.15, elastic 3.21, against
// 1.58 / 4.23 with two warps and no register cap: 200+ registers leave five warps per SM)
template <int N>
constexpr int rpt_min_ctas() { return N <= 2 ? 8 : 12; }

__device__ __forceinline__ void rpt_cp_async4(void *smem, const void *gmem) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"((uint32_t)__cvta_generic_to_shared(smem)), "l"(gmem) : "memory");
}
__device__ __forceinline__ void rpt_cp_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NKEEP>
__device__ __forceinline__ void rpt_cp_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NKEEP) : "memory"); }

template <int MODEL, int N, int MODE>
__global__ void __launch_bounds__(Rpt<MODEL, N>::WARPS * 32, rpt_min_ctas<N>()) rpt_stage_kernel(const StageParams p) {
  using C = Rpt<MODEL, N>;
  constexpr int NP = C::NP, NFP = C::NFP, NFACE = C::NFACE, NF = C::NF, NGEO = C::NGEO;
  constexpr int EPW = C::EPW, NPP = C::NPP, FP = C::FP, TPL = C::TPL, VW = C::VW;
  using Vec = typename RptVec<VW>::T;
  // per warp: two slots of {fields, geometric records, connectivity} (the next tile lands while this one is worked on)
  // and one tile of penalty terms
  __shared__ float s_qt[C::WARPS][2][32 * NPP];
  __shared__ float s_gt[C::WARPS][2][EPW * C::GP];
  __shared__ int s_ct[C::WARPS][2][EPW * 5];                             // nbr [EPW][4], then fcode [EPW] (four bytes each)
  __shared__ float s_ft[C::WARPS][32 * FP];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int ntiles = (p.K - p.kbeg + EPW - 1) / EPW;
  const int nwarps = gridDim.x * C::WARPS;
  float *sf = s_ft[w];

  // tile -> slot, asynchronously (cp.async, 4 bytes each: the tiles have odd row pitches); one group per tile
  auto issue = [&](int tile, int slot) {
    const int ke0 = p.kbeg + tile * EPW;
    const int nel = min(EPW, p.K - ke0);
    {
      const float *src = p.q_in + (size_t)ke0 * NF * NP;               // one contiguous run of nel Nf Np values
      float *dst = s_qt[w][slot];
#pragma unroll
      for (int it = 0; it < (EPW * NF * NP + 31) / 32; ++it) {
        const int idx = it * 32 + lane;
        if (idx < nel * NF * NP) rpt_cp_async4(dst + idx + idx / NP * (NPP - NP), src + idx);
      }
    }
    {
      const float *src = p.geo + (size_t)ke0 * NGEO;
      float *dst = s_gt[w][slot];
#pragma unroll
      for (int it = 0; it < (EPW * NGEO + 31) / 32; ++it) {
        const int idx = it * 32 + lane;
        if (idx < nel * NGEO) rpt_cp_async4(dst + idx + idx / NGEO * (C::GP - NGEO), src + idx);
      }
    }
    {
      int *dst = s_ct[w][slot];
#pragma unroll
      for (int it = 0; it < (EPW * 5 + 31) / 32; ++it) {
        const int idx = it * 32 + lane;
        if (idx < nel * 4) rpt_cp_async4(dst + idx, p.nbr + (size_t)ke0 * 4 + idx);
        else if (idx >= EPW * 4 && idx < EPW * 4 + nel)
          rpt_cp_async4(dst + idx, reinterpret_cast<const int *>(p.fcode) + ke0 + (idx - EPW * 4));
      }
    }
    rpt_cp_commit();
  };

  int tile = blockIdx.x * C::WARPS + w;
  if (tile < ntiles) issue(tile, 0);
#pragma unroll 1
  for (int it = 0; tile < ntiles; tile += nwarps, ++it) {
  const int slot = it & 1;
  if (tile + nwarps < ntiles) {
    issue(tile + nwarps, slot ^ 1);
    rpt_cp_wait<1>();
  } else {
    rpt_cp_wait<0>();
  }
  __syncwarp();                                                          // (this tile's slot is complete, for every lane)
  const int ke0 = p.kbeg + tile * EPW;
  const int nel = min(EPW, p.K - ke0);
  const float *sq = s_qt[w][slot], *sg = s_gt[w][slot];
  const int *sc = s_ct[w][slot];

  // lanes without a row (elastic: 27 of 32; ragged last warp) follow row 0 and store nothing
  const bool valid = lane < nel * NF;
  const int row = valid ? lane : 0;
  const int el = row / NF, f = row - el * NF;
  const int k = ke0 + el;
  const float *g = sg + el * C::GP;
  const size_t base = ((size_t)k * NF + f) * NP;

  // (Copying the whole element behind every face of the tile into shared memory with 16-byte cp.async and reading the traces
  // from there -- 10 wide copies instead of 24 scattered 4-byte loads per tile at acoustic N = 2 -- was measured: 0.72 ->
  // 0.96 ms per stage, elastic 1.89 -> 2.54: it moves 1.7x the bytes through L1 and costs a resident CTA per SM.)
  // ---- exterior traces of this lane's share of the element's face nodes (row a4): every load is issued here, without
  // a branch in between, so that the chain neighbour node -> values is in flight behind the volume term (a lane with no
  // task at t, or a boundary face, reads a valid address and ignores the value)
  constexpr int TG = TPL * NF <= 48 ? TPL : 48 / NF;     // tasks whose traces are fetched ahead (register budget)
  int nbt[TPL];
  float up[TG][NF];
#pragma unroll
  for (int t = 0; t < TPL; ++t) {
    const int j = min(f + NF * t, NFACE - 1), face = j / NFP;
    nbt[t] = sc[el * 4 + face];
  }
  auto fetch = [&](int t, float (&x)[NF]) {
    const int j = min(f + NF * t, NFACE - 1), face = j / NFP, i = j - face * NFP;
    const int code = (sc[EPW * 4 + el] >> (8 * face)) & 255;
    const int nn = __ldg(p.nbrnode + (face * 24 + code) * NFP + i);
    const float *qp = p.q_in + (size_t)(nbt[t] >= 0 ? nbt[t] : k) * NF * NP + nn;
#pragma unroll
    for (int c = 0; c < NF; ++c) x[c] = __ldg(qp + c * NP);
  };
  if (!p.pflux) {
#pragma unroll
    for (int t = 0; t < TG; ++t) fetch(t, up[t]);
  }
  // the residual of this row (LSRK stage with A_s != 0): fetched here, used in the update
  // (bringing the residual rows in with the tile through cp.async instead was measured: acoustic N = 2 0.685 -> 0.738 ms)
  constexpr bool RESPF = MODE == MODE_STAGE;
  float ores[RESPF ? NP : 1];
  if (RESPF && p.a != 0.f) {
#pragma unroll
    for (int n = 0; n < NP; n += VW) {
      const Vec v = *reinterpret_cast<const Vec *>(p.res + base + n);
      if constexpr (VW == 4) { ores[n] = v.x; ores[n + 1] = v.y; ores[n + 2] = v.z; ores[n + 3] = v.w; }
      else if constexpr (VW == 2) { ores[n] = v.x; ores[n + 1] = v.y; }
      else { ores[n] = v; }
    }
  }

  // ---- volume term (rows a1-a3)
  float cf[3][3];
  int src[3], nsrc;
  row_coefficients_s<MODEL>(g, f, cf, src, nsrc);
  // the element's material constants in registers (the penalty terms below read them per face node; the stores to the
  // penalty tile in between keep the compiler from holding shared-memory values across tasks)
  float gm[14];
#pragma unroll
  for (int i = 9; i < 14; ++i) gm[i] = g[i];
  const float *gpen = gm;                                               // (acoustic N = 2: 0.684 -> 0.673 ms per stage)
  const float *own = sq + row * NPP;
  // mean of the four vertex values of the row: D_j 1 = 0, so the shift is exact and removes the cancellation
  const float mean_own = 0.25f * ((own[0] + own[N]) + (own[NFP - 1] + own[NP - 1]));
  const float *sp[3];
  float mean[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    sp[i] = sq + (el * NF + src[i]) * NPP;
    mean[i] = __shfl_sync(0xffffffffu, mean_own, el * NF + src[i]);
  }
  // the row's accumulators as register pairs: an operator pair (n, n + 1) comes from the constant bank as one uniform
  // 64-bit operand, and FFMA2 (the packed FP32 FMA of sm_100) does two nodes per issue slot: half the FMA instructions
  static_assert(NP % 2 == 0, "row accumulators are paired");
  float2 r2[NP / 2];
#pragma unroll
  for (int n = 0; n < NP / 2; ++n) r2[n] = make_float2(0.f, 0.f);
#pragma unroll
  for (int m = 0; m < NP; ++m) {
    const float u0 = sp[0][m] - mean[0], u1 = sp[1][m] - mean[1], u2 = sp[2][m] - mean[2];
    float a[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) a[j] = cf[j][0] * u0 + cf[j][1] * u1 + cf[j][2] * u2;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      const float2 aa = make_float2(a[j], a[j]);
#pragma unroll
      for (int n = 0; n < NP / 2; ++n)
        r2[n] = __ffma2_rn(make_float2(c_rpt_D[(3 * m + j) * NP + 2 * n], c_rpt_D[(3 * m + j) * NP + 2 * n + 1]), aa, r2[n]);
    }
  }

  // ---- surface term (row a5): penalty terms of this lane's face nodes -> tile
#pragma unroll
  for (int t = 0; t < TPL; ++t) {
    const int j = f + NF * t;
    float upl[NF];
    if (t >= TG && !p.pflux) fetch(t, upl);                              // (beyond the register budget: fetched here)
    if (j < NFACE) {
      const int face = j / NFP;
      float F[NF];
      if (p.pflux) {                                                     // interface-centric surface step: terms from the face buffer
#pragma unroll
        for (int c = 0; c < NF; ++c) F[c] = __ldg(p.pflux + ((size_t)k * NF + c) * NFACE + j);
      } else {
        const int nm = __ldg(p.fmask + j);
        const int nb = nbt[t];
        float um[NF], ue[NF];
#pragma unroll
        for (int c = 0; c < NF; ++c) {
          um[c] = sq[(el * NF + c) * NPP + nm];
          ue[c] = t < TG ? up[t < TG ? t : 0][c] : upl[c];
        }
        constexpr int FO = MODEL == 0 ? 12 : 16, FS = MODEL == 0 ? 5 : 8;
        const float *fg = g + FO + FS * face;
        const float nx = fg[0], ny = fg[1], nz = fg[2];
        if (MODEL == 0) {
          float dp, dvn;
          if (nb >= 0) {
            dp = ue[0] - um[0];
            dvn = (ue[1] - um[1]) * nx + (ue[2] - um[2]) * ny + (ue[3] - um[3]) * nz;
          } else {
            acoustic_boundary_jump(nb, um[0], um[1] * nx + um[2] * ny + um[3] * nz, dp, dvn);
          }
          const float4 Pn = acoustic_penalty(gpen, fg, dp, dvn);
          F[0] = Pn.x; F[1] = Pn.y; F[2] = Pn.z; F[3] = Pn.w;
        } else {
          float Tmx, Tmy, Tmz;
          traction(um, nx, ny, nz, Tmx, Tmy, Tmz);
          float dv[3], dT[3];
          if (nb >= 0) {
            float Tpx, Tpy, Tpz;
            traction(ue, nx, ny, nz, Tpx, Tpy, Tpz);
            dv[0] = ue[0] - um[0]; dv[1] = ue[1] - um[1]; dv[2] = ue[2] - um[2];
            dT[0] = Tpx - Tmx; dT[1] = Tpy - Tmy; dT[2] = Tpz - Tmz;
          } else {
            elastic_boundary_jump(nb, um, Tmx, Tmy, Tmz, nx, ny, nz, dv, dT);
          }
          elastic_penalty(gpen, fg, dv, dT, F);
        }
      }
#pragma unroll
      for (int c = 0; c < NF; ++c) sf[(el * NF + c) * FP + j] = F[c];
    }
  }
  __syncwarp();

  // ---- lift (row a6): this lane's field
  {
    const float *fr = sf + row * FP;
#pragma unroll
    for (int j = 0; j < NFACE; ++j) {
      const float2 Fj = make_float2(fr[j], fr[j]);
#pragma unroll
      for (int n = 0; n < NP / 2; ++n) r2[n] = __ffma2_rn(make_float2(c_rpt_L[j * NP + 2 * n], c_rpt_L[j * NP + 2 * n + 1]), Fj, r2[n]);
    }
  }
  float r[NP];
#pragma unroll
  for (int n = 0; n < NP / 2; ++n) { r[2 * n] = r2[n].x; r[2 * n + 1] = r2[n].y; }
  // ---- LSRK update (row a7).  Results leave through the tiles: a lane's row in global memory is Np floats at a stride of
  // Np floats -- a vector store per lane touches one line per row, ten lines per instruction at N = 2 -- while the warp's
  // rows together are one contiguous run.  So each lane writes its new q row over its (now unused) row of the field slot
  // and its residual / right-hand side over its row of the penalty tile, and the warp copies both out line by line.
  // (same-box A/B, ms per stage: acoustic N = 2 0.723 -> 0.684, N = 3 1.29 -> 1.08; the elastic tiles -- 27 rows -- and N = 1
  // gain no lines and pay the extra shared-memory traffic: elastic N = 2 1.90 -> 1.97, acoustic N = 1 0.87 -> 0.93: direct there)
  constexpr bool COUT = MODEL == 0 && N >= 2;
  float *sqw = s_qt[w][slot] + row * NPP;                                // this lane's row of the field slot
  float *sfw = sf + row * FP;                                            // and of the penalty tile
  auto ldv = [&](const float *ptr, int n, float (&x)[VW]) {
    const Vec v = *reinterpret_cast<const Vec *>(ptr + n);
    if constexpr (VW == 4) { x[0] = v.x; x[1] = v.y; x[2] = v.z; x[3] = v.w; }
    else if constexpr (VW == 2) { x[0] = v.x; x[1] = v.y; }
    else { x[0] = v; }
  };
  auto stv = [&](float *gptr, float *srow, int n, const float (&x)[VW]) {
    if (COUT) {
#pragma unroll
      for (int t = 0; t < VW; ++t) srow[n + t] = x[t];
    } else {
      Vec v;
      if constexpr (VW == 4) v = make_float4(x[0], x[1], x[2], x[3]);
      else if constexpr (VW == 2) v = make_float2(x[0], x[1]);
      else v = x[0];
      *reinterpret_cast<Vec *>(gptr + n) = v;
    }
  };
  if (valid) {
#pragma unroll
  for (int n = 0; n < NP; n += VW) {
    float rr[VW], qq[VW];
#pragma unroll
    for (int t = 0; t < VW; ++t) { rr[t] = r[n + t]; qq[t] = own[n + t]; }
    if (MODE == MODE_RHS) {
      stv(p.rhs + base, sfw, n, rr);
    } else if (MODE == MODE_AB3) {
      float x[VW], y[VW];
      ldv(p.res + base, n, x);
      ldv(p.hist2 + base, n, y);
      stv(p.rhs + base, sfw, n, rr);
#pragma unroll
      for (int t = 0; t < VW; ++t) qq[t] = fmaf(p.b, y[t], fmaf(p.a, x[t], fmaf(p.dt, rr[t], qq[t])));
      stv(p.q_out + base, sqw, n, qq);
    } else {
      float rs[VW];
#pragma unroll
      for (int t = 0; t < VW; ++t) rs[t] = p.dt * rr[t];
      if (p.a != 0.f) {
        float o[VW];
        if (RESPF) {
#pragma unroll
          for (int t = 0; t < VW; ++t) o[t] = ores[RESPF ? n + t : 0];
        } else {
          ldv(p.res + base, n, o);
        }
#pragma unroll
        for (int t = 0; t < VW; ++t) rs[t] = fmaf(p.a, o[t], rs[t]);
      }
      stv(p.res + base, sfw, n, rs);
#pragma unroll
      for (int t = 0; t < VW; ++t) qq[t] = fmaf(p.b, rs[t], qq[t]);
      stv(p.q_out + base, sqw, n, qq);
    }
  }
  }
  if (COUT) {
    __syncwarp();
    const int total = nel * NF * NP;
    const size_t g0 = (size_t)ke0 * NF * NP;
    float *gr = (MODE == MODE_STAGE ? p.res : p.rhs) + g0;               // what the penalty tile carries
    const float *sqt = s_qt[w][slot];
#pragma unroll
    for (int i = 0; i < (EPW * NF * NP + 31) / 32; ++i) {
      const int idx = i * 32 + lane;
      if (idx < total) {
        const int rw = idx / NP;
        gr[idx] = sf[idx + rw * (FP - NP)];
        if (MODE != MODE_RHS) p.q_out[g0 + idx] = sqt[idx + rw * (NPP - NP)];
      }
    }
  }
  __syncwarp();                                                          // (every lane is done with this slot and the penalty tile)
  }
}

}  // namespace dgk
