// Interface-centric surface step of libdg (optional, dg_options.surface = 1): the surface kernel of the paper's SGEMM
// strategy -- "the surface kernel iterates over all the interfaces of the mesh.  Each thread computes the numerical
// fluxes corresponding to one face node for both sides of the interface" (section 3.3) -- as an
// alternative producer of the penalty terms (rows a4 + a5): one thread per (interface, face node) gathers the two
// traces once, evaluates the upwind penalty terms of both elements (each with its own outward normal, g^sur and
// materials, PAPER.md:45-51 / 71-84) and writes them, already multiplied by g^sur, into the face buffer
//     pflux[K][Nfields][4 Nfp]        (the P^p, P^v arrays of PAPER.md:206-209 in one),
// from which the stage kernels then lift (row a6) instead of gathering themselves.  Boundary faces (no neighbour) are
// handled by the threads behind the interior ones with the mirror states of DESIGN.md reading Q9.
// Cost against the element-centric default: half the gathers and jump evaluations, but one extra write + read of
// Nfields 4 Nfp floats per element through HBM (profiles/r02_interface_ab.md has the measured A/B).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "flux.cuh"
#include "kernels.cuh"

namespace dgk {

struct IfaceParams {
  const float *__restrict__ q;                 // [K][Nf][pitch]
  float *__restrict__ pflux;                   // [K][Nf][4 Nfp]
  const float *__restrict__ geo;               // [K][GEO_*]
  const int *__restrict__ nbr;                 // [K][4] neighbour element or -(bc tag)
  const unsigned char *__restrict__ fcode;     // [K][4] neighbour face * 6 + vertex correspondence
  const int *__restrict__ faces;               // [nint] owner faces 4 k + f of the interior interfaces, then [nbnd] boundary faces
  const unsigned short *__restrict__ fmask;    // [4 Nfp]
  const unsigned short *__restrict__ nbrnode;  // [4][24][Nfp] neighbour's volume node
  const unsigned short *__restrict__ nbrface;  // [4][24][Nfp] its index on the neighbour's face
  int nint, nbnd, pitch;
};

template <int MODEL, int N>
__global__ void __launch_bounds__(256) iface_flux_kernel(const IfaceParams p) {
  using D = Deg<N>;
  constexpr int NFP = D::NFP, NFACE = D::NFACE;
  constexpr int NF = MODEL == 0 ? 4 : 9, NGEO = MODEL == 0 ? GEO_AC : GEO_EL;
  constexpr int FO = MODEL == 0 ? 12 : 16, FS = MODEL == 0 ? 5 : 8;     // face records inside the element record
  const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int face = (int)(t / NFP), i = (int)(t - (long long)face * NFP);
  if (face >= p.nint + p.nbnd) return;
  const int fa = __ldg(p.faces + face);
  const int k = fa >> 2, f = fa & 3;
  const int nm = __ldg(p.fmask + f * NFP + i);
  const float *gA = p.geo + (size_t)k * NGEO, *fgA = gA + FO + FS * f;
  const float *qa = p.q + ((size_t)k * NF) * p.pitch + nm;
  float ua[NF], FA[NF];
#pragma unroll
  for (int c = 0; c < NF; ++c) ua[c] = __ldg(qa + (size_t)c * p.pitch);
  float *outA = p.pflux + ((size_t)k * NF) * NFACE + f * NFP + i;
  const int nb = __ldg(p.nbr + fa);
  if (nb < 0) {                                  // boundary face: mirror state
    if (MODEL == 0) {
      float dp, dvn;
      acoustic_boundary_jump(nb, ua[0], ua[1] * fgA[0] + ua[2] * fgA[1] + ua[3] * fgA[2], dp, dvn);
      const float4 P = acoustic_penalty(gA, fgA, dp, dvn);
      FA[0] = P.x; FA[1] = P.y; FA[2] = P.z; FA[3] = P.w;
    } else {
      float Tx, Ty, Tz, dv[3], dT[3];
      traction(ua, fgA[0], fgA[1], fgA[2], Tx, Ty, Tz);
      elastic_boundary_jump(nb, ua, Tx, Ty, Tz, fgA[0], fgA[1], fgA[2], dv, dT);
      elastic_penalty(gA, fgA, dv, dT, FA);
    }
#pragma unroll
    for (int c = 0; c < NF; ++c) outA[(size_t)c * NFACE] = FA[c];
    return;
  }
  // interior interface: the neighbour's side is computed by this thread as well
  const int code = (int)__ldg(p.fcode + fa), g = code / 6;
  const int tab = (f * 24 + code) * NFP + i;
  const int nn = __ldg(p.nbrnode + tab), ii = __ldg(p.nbrface + tab);
  const float *gB = p.geo + (size_t)nb * NGEO, *fgB = gB + FO + FS * g;
  const float *qb = p.q + ((size_t)nb * NF) * p.pitch + nn;
  float ub[NF], FB[NF];
#pragma unroll
  for (int c = 0; c < NF; ++c) ub[c] = __ldg(qb + (size_t)c * p.pitch);
  if (MODEL == 0) {
    {
      const float dp = ub[0] - ua[0];
      const float dvn = (ub[1] - ua[1]) * fgA[0] + (ub[2] - ua[2]) * fgA[1] + (ub[3] - ua[3]) * fgA[2];
      const float4 P = acoustic_penalty(gA, fgA, dp, dvn);
      FA[0] = P.x; FA[1] = P.y; FA[2] = P.z; FA[3] = P.w;
    }
    {
      const float dp = ua[0] - ub[0];
      const float dvn = (ua[1] - ub[1]) * fgB[0] + (ua[2] - ub[2]) * fgB[1] + (ua[3] - ub[3]) * fgB[2];
      const float4 P = acoustic_penalty(gB, fgB, dp, dvn);
      FB[0] = P.x; FB[1] = P.y; FB[2] = P.z; FB[3] = P.w;
    }
  } else {
    {
      float Tmx, Tmy, Tmz, Tpx, Tpy, Tpz;
      traction(ua, fgA[0], fgA[1], fgA[2], Tmx, Tmy, Tmz);
      traction(ub, fgA[0], fgA[1], fgA[2], Tpx, Tpy, Tpz);
      const float dv[3] = {ub[0] - ua[0], ub[1] - ua[1], ub[2] - ua[2]};
      const float dT[3] = {Tpx - Tmx, Tpy - Tmy, Tpz - Tmz};
      elastic_penalty(gA, fgA, dv, dT, FA);
    }
    {
      float Tmx, Tmy, Tmz, Tpx, Tpy, Tpz;
      traction(ub, fgB[0], fgB[1], fgB[2], Tmx, Tmy, Tmz);
      traction(ua, fgB[0], fgB[1], fgB[2], Tpx, Tpy, Tpz);
      const float dv[3] = {ua[0] - ub[0], ua[1] - ub[1], ua[2] - ub[2]};
      const float dT[3] = {Tpx - Tmx, Tpy - Tmy, Tpz - Tmz};
      elastic_penalty(gB, fgB, dv, dT, FB);
    }
  }
  float *outB = p.pflux + ((size_t)nb * NF) * NFACE + g * NFP + ii;
#pragma unroll
  for (int c = 0; c < NF; ++c) {
    outA[(size_t)c * NFACE] = FA[c];
    outB[(size_t)c * NFACE] = FB[c];
  }
}

}  // namespace dgk
