// Upwind penalty terms of the hot path (row a5), shared by every stage-kernel variant of libdg.
// Inputs are the jumps (exterior minus interior trace) at one face node; outputs are the penalty
// vectors already multiplied by g^sur, ready to be lifted (r += LIFT * F).
//   acoustic: PAPER.md:45-51; elastic: PAPER.md:71-84; boundary mirror states: DESIGN.md reading Q9.
// Per-element record `g` and per-face record `fg` are laid out as in kernels.cuh (GEO_AC / GEO_EL).
#pragma once
#include <cuda_runtime.h>

namespace dgk {

constexpr int GEO_AC = 32;   // floats per element, acoustic: G[9] kappa 1/rho c | 4 x (nx ny nz fk Z+)
constexpr int GEO_EL = 48;   // elastic: G[9] 1/rho lam mu cp cs pad pad | 4 x (nx ny nz fkp fks Zp+ Zs+ pad)

// ---- acoustic ------------------------------------------------------------------------------------
// jumps for a face without neighbour: nb = -(bc tag).  (pm, vnm) = interior pressure and normal velocity
__device__ __forceinline__ void acoustic_boundary_jump(int nb, float pm, float vnm, float &dp, float &dvn) {
  if (nb == -2) {            // free (pressure release): p+ = -p-, v+ = v-
    dp = -2.f * pm;
    dvn = 0.f;
  } else {                   // rigid / slip: p+ = p-, v_n+ = -v_n-
    dp = 0.f;
    dvn = -2.f * vnm;
  }
}

// fg = (nx ny nz fk Z+) with fk = g^sur k_c / 2;  F = (-g^sur p_p, -g^sur p_v)
__device__ __forceinline__ float4 acoustic_penalty(const float *g, const float *fg, float dp, float dvn) {
  const float sc = fg[3] * (dp - fg[4] * dvn);     // g^sur k_c alpha_c
  const float kap = g[9], cc = g[11];
  const float t = -cc * sc;
  return make_float4(kap * sc, t * fg[0], t * fg[1], t * fg[2]);
}

// ---- elastic -------------------------------------------------------------------------------------
// interior traction T- = sigma- n from the nine interior values um (vx vy vz sxx syy szz sxy sxz syz)
__device__ __forceinline__ void traction(const float *u, float nx, float ny, float nz, float &Tx, float &Ty, float &Tz) {
  Tx = u[3] * nx + u[6] * ny + u[7] * nz;
  Ty = u[6] * nx + u[4] * ny + u[8] * nz;
  Tz = u[7] * nx + u[8] * ny + u[5] * nz;
}

__device__ __forceinline__ void elastic_boundary_jump(int nb, const float *um, float Tmx, float Tmy, float Tmz, float nx, float ny,
                                                      float nz, float *dv, float *dT) {
  if (nb == -1) {            // rigid: v+ = -v-, T+ = T-
    dv[0] = -2.f * um[0]; dv[1] = -2.f * um[1]; dv[2] = -2.f * um[2];
    dT[0] = dT[1] = dT[2] = 0.f;
  } else if (nb == -2) {     // free surface: T+ = -T-, v+ = v-
    dv[0] = dv[1] = dv[2] = 0.f;
    dT[0] = -2.f * Tmx; dT[1] = -2.f * Tmy; dT[2] = -2.f * Tmz;
  } else {                   // slip: v_n+ = -v_n-, T_t+ = -T_t-
    const float vn = um[0] * nx + um[1] * ny + um[2] * nz;
    const float Tn = Tmx * nx + Tmy * ny + Tmz * nz;
    dv[0] = -2.f * vn * nx; dv[1] = -2.f * vn * ny; dv[2] = -2.f * vn * nz;
    dT[0] = -2.f * (Tmx - Tn * nx); dT[1] = -2.f * (Tmy - Tn * ny); dT[2] = -2.f * (Tmz - Tn * nz);
  }
}

// fg = (nx ny nz fkp fks Zp+ Zs+) with fkp = g^sur k_p / 2, fks = g^sur k_s / 2 (they absorb the halves of
// the semi-jumps);  F[0..2] = g^sur p_v, F[3..8] = g^sur P_sigma (xx yy zz xy xz yz)
__device__ __forceinline__ void elastic_penalty(const float *g, const float *fg, const float *dv, const float *dT, float *F) {
  const float nx = fg[0], ny = fg[1], nz = fg[2], fkp = fg[3], fks = fg[4], Zpp = fg[5], Zsp = fg[6];
  const float dTn = dT[0] * nx + dT[1] * ny + dT[2] * nz;
  const float dvn = dv[0] * nx + dv[1] * ny + dv[2] * nz;
  const float kpa = fkp * (dTn + Zpp * dvn);                    // g^sur k_p alpha_p
  const float asx = fks * (dT[0] + Zsp * dv[0]), asy = fks * (dT[1] + Zsp * dv[1]), asz = fks * (dT[2] + Zsp * dv[2]);
  const float ksa = asx * nx + asy * ny + asz * nz;             // g^sur k_s alpha_s
  const float lam = g[10], mu = g[11], cp = g[12], cs = g[13];
  const float cn = kpa * cp - ksa * cs;
  F[0] = cn * nx + cs * asx;
  F[1] = cn * ny + cs * asy;
  F[2] = cn * nz + cs * asz;
  const float d0 = kpa * lam, d1 = 2.f * mu * (kpa - ksa);
  F[3] = d0 + d1 * nx * nx + 2.f * mu * nx * asx;
  F[4] = d0 + d1 * ny * ny + 2.f * mu * ny * asy;
  F[5] = d0 + d1 * nz * nz + 2.f * mu * nz * asz;
  F[6] = d1 * nx * ny + mu * (nx * asy + ny * asx);
  F[7] = d1 * nx * nz + mu * (nx * asz + nz * asx);
  F[8] = d1 * ny * nz + mu * (ny * asz + nz * asy);
}

}  // namespace dgk
