// Fused SIMT stage kernels of libdg (sm_100a).  One launch evaluates, for a batch of G*E elements per
// CTA, every row of the hot path: volume pre-combination (a1), the three
// differentiation mat-vecs per field (a2), post-combination (a3), face gather through the compressed
// connectivity (a4), upwind penalty terms (a5), merged lift (a6) and the LSRK update (a7).
//
// Mapping ("one node per thread, E elements per thread"): thread t owns output node n = t % Np of the
// E elements of node-group g = t / Np; operator columns D_j[n][m], L[n][j] stream through L1 as
// coalesced loads (they are shared by every CTA on the SM), the per-element inputs are staged in shared
// memory as float4 so that one broadcast LDS.128 feeds 4-6 FFMAs.  Prior art for the thread-per-node
// idea: PAPER.md:175 and Table 2; the register blocking over elements, the fused surface/update and
// the compressed connectivity are this build's.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "flux.cuh"

namespace dgk {

// MODE_AB3: the paper's own update (eq. (4)) as the epilogue: rhs <- r(q_in) (the new r^m),
// q_out <- q_in + dt r^m + a res + b hist2 with res = r^{m-1}, hist2 = r^{m-2} (read only) and dt, a, b = dt (23, -16, 5) / 12
enum { MODE_RHS = 0, MODE_STAGE = 1, MODE_AB3 = 2 };

struct StageParams {
  const float *__restrict__ q_in;
  float *__restrict__ q_out;
  float *__restrict__ res;
  float *__restrict__ rhs;
  const float *__restrict__ hist2;           // MODE_AB3: r^{m-2}
  const float *__restrict__ pflux;           // interface-centric surface step (iface_kernels.cuh): [K][Nf][4 Nfp] penalty terms
                                             // times g^sur, computed beforehand; NULL = gather and evaluate them here
  const float *__restrict__ DT;              // [3][Np][Np]  DT[d][m][n] = D_d[n][m]
  const float *__restrict__ LT;              // [4Nfp][Np]   LT[j][n]    = LIFT[n][j]
  const float *__restrict__ geo;             // [K][GEO_*]
  const int *__restrict__ nbr;               // [K][4] neighbour element or -(bc tag)
  const unsigned char *__restrict__ fcode;   // [K][4] g*6+s
  const unsigned short *__restrict__ fmask;  // [4Nfp]
  const unsigned short *__restrict__ nbrnode;  // [4][24][Nfp]
  int K;                                     // end of the element range this launch works on (all elements: K)
  int kbeg;                                  // first element of the range (dg_stage_range; 0 otherwise)
  int G;                                     // node groups per CTA
  float a, b, dt;                            // LSRK A_s, B_s, dt
};

template <int N>
struct Deg {
  static constexpr int NP = (N + 1) * (N + 2) * (N + 3) / 6;
  static constexpr int NFP = (N + 1) * (N + 2) / 2;
  static constexpr int NFACE = 4 * NFP;
};

// shared-memory floats per element of the batch
template <int MODEL, int N>
struct Smem {
  static constexpr int NF = MODEL == 0 ? 4 : 9;
  static constexpr int NGEO = MODEL == 0 ? GEO_AC : GEO_EL;
  static constexpr int VIN4 = MODEL == 0 ? 1 : 3;   // float4 per node of packed volume input
  static constexpr int FLX4 = MODEL == 0 ? 1 : 3;   // float4 per face node of penalty terms
  static constexpr int PER_ELEM = NGEO + 8 + NF * Deg<N>::NP + 4 * VIN4 * Deg<N>::NP + 4 * FLX4 * Deg<N>::NFACE;
  static size_t bytes(int EB) { return (size_t)EB * PER_ELEM * 4 + 16; }
};

// ------------------------------------------------------------------------------------------------
template <int MODEL, int N, int E, int MODE>
__global__ void stage_kernel(const StageParams p) {
  using D = Deg<N>;
  using S = Smem<MODEL, N>;
  constexpr int NP = D::NP, NFP = D::NFP, NFACE = D::NFACE, NF = S::NF, NGEO = S::NGEO;
  const int EB = p.G * E;
  const int NT = blockDim.x;
  const int tid = threadIdx.x;
  const int k0 = p.kbeg + blockIdx.x * EB;
  const int nvalid = min(EB, p.K - k0);

  extern __shared__ float4 smem4[];
  float4 *s_vin = smem4;                                   // [EB][NP][VIN4]
  float4 *s_flux = s_vin + (size_t)EB * NP * S::VIN4;      // [EB][NFACE][FLX4]
  float *s_q = (float *)(s_flux + (size_t)EB * NFACE * S::FLX4);   // [EB][NF][NP]
  float *s_geo = s_q + (size_t)EB * NF * NP;               // [EB][NGEO]
  int *s_nbr = (int *)(s_geo + (size_t)EB * NGEO);         // [EB][4]
  int *s_code = s_nbr + EB * 4;                            // [EB][4]

  // ---- phase 0: per-element constants and the raw fields of the batch
  for (int i = tid; i < EB * NGEO; i += NT) s_geo[i] = (i < nvalid * NGEO) ? p.geo[(size_t)k0 * NGEO + i] : 0.f;
  for (int i = tid; i < EB * 4; i += NT) {
    const bool ok = i < nvalid * 4;
    s_nbr[i] = ok ? p.nbr[(size_t)k0 * 4 + i] : -1;
    s_code[i] = ok ? (int)p.fcode[(size_t)k0 * 4 + i] : 0;
  }
  {
    // the batch's fields are one contiguous run of nvalid*NF*NP floats
    const float *src = p.q_in + (size_t)k0 * NF * NP;
    const int nload = nvalid * NF * NP;
    for (int i = tid; i < EB * NF * NP; i += NT) s_q[i] = (i < nload) ? __ldg(src + i) : 0.f;
  }
  __syncthreads();

  // ---- phase A: pre-combine the divergence inputs (row a1).  Every input of a differentiation is
  // shifted by the mean of the element's four vertex values: D_j 1 = 0, so the result is unchanged in
  // exact arithmetic, while the fp32 products, the partial sums and the effect of the operators' own
  // fp32 rounding shrink from O(|q|) to O(h |grad q|).
  for (int it = tid; it < EB * NP; it += NT) {
    const int e = it / NP, m = it - e * NP;
    const float *g = s_geo + e * NGEO;
    const float *qe = s_q + e * NF * NP;
    float u[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const float *qf = qe + f * NP;
      u[f] = qf[m] - 0.25f * ((qf[0] + qf[N]) + (qf[NFP - 1] + qf[NP - 1]));   // minus the mean of the 4 vertex values
    }
    if (MODEL == 0) {
      // eq. (5): w_j = sum_i g_ij v_i
      float4 w;
      w.x = u[0];
      w.y = g[0] * u[1] + g[3] * u[2] + g[6] * u[3];
      w.z = g[1] * u[1] + g[4] * u[2] + g[7] * u[3];
      w.w = g[2] * u[1] + g[5] * u[2] + g[8] * u[3];
      s_vin[it] = w;
    } else {
      // w_{i,n} = sum_m g_mn sigma_im ; fields vx vy vz sxx syy szz sxy sxz syz
      const float sg[3][3] = {{u[3], u[6], u[7]}, {u[6], u[4], u[8]}, {u[7], u[8], u[5]}};
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        float4 w;
        w.x = u[i];
        w.y = g[0] * sg[i][0] + g[3] * sg[i][1] + g[6] * sg[i][2];
        w.z = g[1] * sg[i][0] + g[4] * sg[i][1] + g[7] * sg[i][2];
        w.w = g[2] * sg[i][0] + g[5] * sg[i][1] + g[8] * sg[i][2];
        s_vin[it * 3 + i] = w;
      }
    }
  }

  // ---- phase B: face gather (a4) and penalty terms times g^sur (a5)
  for (int it = tid; it < EB * NFACE; it += NT) {
    const int e = it / NFACE, j = it - e * NFACE;
    const int f = j / NFP, i = j - f * NFP;
    const float *g = s_geo + e * NGEO;
    if (p.pflux) {                              // penalty terms from the face buffer
      const float *src = p.pflux + ((size_t)(k0 + e) * NF) * NFACE + j;
      const bool ok = e < nvalid;
      float F[NF];
#pragma unroll
      for (int c = 0; c < NF; ++c) F[c] = ok ? __ldg(src + (size_t)c * NFACE) : 0.f;
      if (MODEL == 0) {
        s_flux[it] = make_float4(F[0], F[1], F[2], F[3]);
      } else {
        s_flux[it * 3 + 0] = make_float4(F[0], F[1], F[2], F[3]);
        s_flux[it * 3 + 1] = make_float4(F[4 % NF], F[5 % NF], F[6 % NF], F[7 % NF]);
        s_flux[it * 3 + 2] = make_float4(F[8 % NF], 0.f, 0.f, 0.f);
      }
      continue;
    }
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
      const float4 F = acoustic_penalty(g, fg, dp, dvn);
      s_flux[it] = (e < nvalid) ? F : make_float4(0.f, 0.f, 0.f, 0.f);
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
      float F[9];
      elastic_penalty(g, fg, dv, dT, F);
      const bool ok = e < nvalid;
      s_flux[it * 3 + 0] = ok ? make_float4(F[0], F[1], F[2], F[3]) : make_float4(0.f, 0.f, 0.f, 0.f);
      s_flux[it * 3 + 1] = ok ? make_float4(F[4], F[5], F[6], F[7]) : make_float4(0.f, 0.f, 0.f, 0.f);
      s_flux[it * 3 + 2] = ok ? make_float4(F[8], 0.f, 0.f, 0.f) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
  }
  __syncthreads();

  // ---- phase C: dense contractions (a2, a6) with the post-combination (a3) in registers
  if (tid >= p.G * NP) return;
  const int grp = tid / NP, n = tid - grp * NP;
  const int e0 = grp * E;
  constexpr int NACC = MODEL == 0 ? 4 : 12;
  float acc[E][NACC];
#pragma unroll
  for (int ee = 0; ee < E; ++ee)
#pragma unroll
    for (int c = 0; c < NACC; ++c) acc[ee][c] = 0.f;
  {
    const float *dr_p = p.DT + n, *ds_p = p.DT + NP * NP + n, *dt_p = p.DT + 2 * NP * NP + n;
    const float4 *vin = s_vin + (size_t)e0 * NP * S::VIN4;
#pragma unroll 2
    for (int m = 0; m < NP; ++m) {
      const float dr = __ldg(dr_p + m * NP), ds = __ldg(ds_p + m * NP), dt = __ldg(dt_p + m * NP);
#pragma unroll
      for (int ee = 0; ee < E; ++ee) {
        if (MODEL == 0) {
          const float4 v = vin[ee * NP + m];
          acc[ee][0] = fmaf(dr, v.x, acc[ee][0]);
          acc[ee][1] = fmaf(ds, v.x, acc[ee][1]);
          acc[ee][2] = fmaf(dt, v.x, acc[ee][2]);
          acc[ee][3] = fmaf(dr, v.y, acc[ee][3]);
          acc[ee][3] = fmaf(ds, v.z, acc[ee][3]);
          acc[ee][3] = fmaf(dt, v.w, acc[ee][3]);
        } else {
#pragma unroll
          for (int i = 0; i < 3; ++i) {
            const float4 v = vin[(ee * NP + m) * 3 + i];
            acc[ee][3 * i + 0] = fmaf(dr, v.x, acc[ee][3 * i + 0]);
            acc[ee][3 * i + 1] = fmaf(ds, v.x, acc[ee][3 * i + 1]);
            acc[ee][3 * i + 2] = fmaf(dt, v.x, acc[ee][3 * i + 2]);
            acc[ee][9 + i] = fmaf(dr, v.y, acc[ee][9 + i]);
            acc[ee][9 + i] = fmaf(ds, v.z, acc[ee][9 + i]);
            acc[ee][9 + i] = fmaf(dt, v.w, acc[ee][9 + i]);
          }
        }
      }
    }
  }
  float r[E][NF];
#pragma unroll
  for (int ee = 0; ee < E; ++ee) {
    const float *g = s_geo + (e0 + ee) * NGEO;
    if (MODEL == 0) {
      // eq. (5)-(6)
      const float kap = g[9], irho = g[10];
      r[ee][0] = -kap * acc[ee][3];
#pragma unroll
      for (int i = 0; i < 3; ++i)
        r[ee][1 + i] = -irho * (g[3 * i + 0] * acc[ee][0] + g[3 * i + 1] * acc[ee][1] + g[3 * i + 2] * acc[ee][2]);
    } else {
      const float irho = g[9], lam = g[10], mu = g[11];
      float gv[3][3];   // gv[i][j] = d_j v_i = sum_m g_jm (D_m v_i)
#pragma unroll
      for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j)
          gv[i][j] = g[3 * j + 0] * acc[ee][3 * i + 0] + g[3 * j + 1] * acc[ee][3 * i + 1] + g[3 * j + 2] * acc[ee][3 * i + 2];
      const float div = gv[0][0] + gv[1][1] + gv[2][2];
      r[ee][0] = irho * acc[ee][9];
      r[ee][1] = irho * acc[ee][10];
      r[ee][2] = irho * acc[ee][11];
      r[ee][3] = lam * div + 2.f * mu * gv[0][0];
      r[ee][4] = lam * div + 2.f * mu * gv[1][1];
      r[ee][5] = lam * div + 2.f * mu * gv[2][2];
      r[ee][6] = mu * (gv[0][1] + gv[1][0]);
      r[ee][7] = mu * (gv[0][2] + gv[2][0]);
      r[ee][8] = mu * (gv[1][2] + gv[2][1]);
    }
  }
  {
    const float *l_p = p.LT + n;
    const float4 *flx = s_flux + (size_t)e0 * NFACE * S::FLX4;
#pragma unroll 2
    for (int j = 0; j < NFACE; ++j) {
      const float l = __ldg(l_p + j * NP);
#pragma unroll
      for (int ee = 0; ee < E; ++ee) {
        if (MODEL == 0) {
          const float4 F = flx[ee * NFACE + j];
          r[ee][0] = fmaf(l, F.x, r[ee][0]);
          r[ee][1] = fmaf(l, F.y, r[ee][1]);
          r[ee][2] = fmaf(l, F.z, r[ee][2]);
          r[ee][3] = fmaf(l, F.w, r[ee][3]);
        } else {
          const float4 F0 = flx[(ee * NFACE + j) * 3 + 0], F1 = flx[(ee * NFACE + j) * 3 + 1];
          const float F2 = flx[(ee * NFACE + j) * 3 + 2].x;
          r[ee][0] = fmaf(l, F0.x, r[ee][0]);
          r[ee][1] = fmaf(l, F0.y, r[ee][1]);
          r[ee][2] = fmaf(l, F0.z, r[ee][2]);
          r[ee][3] = fmaf(l, F0.w, r[ee][3]);
          r[ee][4] = fmaf(l, F1.x, r[ee][4]);
          r[ee][5] = fmaf(l, F1.y, r[ee][5]);
          r[ee][6] = fmaf(l, F1.z, r[ee][6]);
          r[ee][7] = fmaf(l, F1.w, r[ee][7]);
          r[ee][8] = fmaf(l, F2, r[ee][8]);
        }
      }
    }
  }
  // ---- phase D: LSRK update (a7) and coalesced stores
#pragma unroll
  for (int ee = 0; ee < E; ++ee) {
    const int e = e0 + ee;
    if (e >= nvalid) break;
    const size_t base = ((size_t)(k0 + e) * NF) * NP + n;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const size_t idx = base + (size_t)f * NP;
      if (MODE == MODE_RHS) {
        p.rhs[idx] = r[ee][f];
      } else if (MODE == MODE_AB3) {
        p.rhs[idx] = r[ee][f];
        p.q_out[idx] = fmaf(p.b, __ldg(p.hist2 + idx), fmaf(p.a, p.res[idx], fmaf(p.dt, r[ee][f], s_q[(e * NF + f) * NP + n])));
      } else {
        float rs = p.dt * r[ee][f];
        if (p.a != 0.f) rs = fmaf(p.a, p.res[idx], rs);
        p.res[idx] = rs;
        p.q_out[idx] = fmaf(p.b, rs, s_q[(e * NF + f) * NP + n]);
      }
    }
  }
}

}  // namespace dgk
