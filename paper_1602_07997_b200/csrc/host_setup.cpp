// Host-side setup of libdg (see host_setup.hpp).  Plain C++17, fp64.
#include "host_setup.hpp"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <numeric>
#include <stdexcept>

namespace dgh {

const int PERMS[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
const int FACE_VERTS[4][3] = {{0, 1, 2}, {0, 1, 3}, {1, 2, 3}, {0, 2, 3}};

namespace {

// ---- classical Jacobi polynomials P_n^{(a,b)} (b >= 0), their norms and derivatives ----------
double jacobi_classical(int n, double a, double b, double x) {
  if (n < 0) return 0.0;
  double p0 = 1.0;
  if (n == 0) return p0;
  double p1 = 0.5 * ((a - b) + (a + b + 2.0) * x);
  for (int k = 1; k < n; ++k) {
    const double s = 2.0 * k + a + b;
    const double c1 = 2.0 * (k + 1) * (k + a + b + 1.0) * s;
    const double c2 = (s + 1.0) * (a * a - b * b);
    const double c3 = s * (s + 1.0) * (s + 2.0);
    const double c4 = 2.0 * (k + a) * (k + b) * (s + 2.0);
    const double p2 = ((c2 + c3 * x) * p1 - c4 * p0) / c1;
    p0 = p1;
    p1 = p2;
  }
  return p1;
}
double jacobi_norm(int n, double a, double b) {   // sqrt of int (1-x)^a (1+x)^b P_n^2
  const double lg = (a + b + 1.0) * std::log(2.0) - std::log(2.0 * n + a + b + 1.0) + std::lgamma(n + a + 1.0) +
                    std::lgamma(n + b + 1.0) - std::lgamma(n + a + b + 1.0) - std::lgamma(n + 1.0);
  return std::exp(0.5 * lg);
}
inline double jac(int n, double a, double x) { return jacobi_classical(n, a, 0.0, x) / jacobi_norm(n, a, 0.0); }
inline double djac(int n, double a, double x) {
  if (n == 0) return 0.0;
  return 0.5 * (n + a + 1.0) * jacobi_classical(n - 1, a + 1.0, 1.0, x) / jacobi_norm(n, a, 0.0);
}

// ---- Gauss-Lobatto-Legendre points: +-1 and the zeros of P_{N-1}^{(1,1)}, Newton with deflation
std::vector<double> gauss_lobatto(int N) {
  std::vector<double> x(N + 1);
  x[0] = -1.0;
  x[N] = 1.0;
  const int ni = N - 1;
  const double pi = std::acos(-1.0);
  for (int k = 0; k < ni; ++k) {
    double z = -std::cos(pi * (k + 1.0) / N);
    for (int it = 0; it < 100; ++it) {
      const double f = jacobi_classical(ni, 1.0, 1.0, z);
      const double df = 0.5 * (ni + 3.0) * jacobi_classical(ni - 1, 2.0, 2.0, z);
      double defl = 0.0;
      for (int j = 0; j < k; ++j) defl += 1.0 / (z - x[1 + j]);
      const double dz = f / (df - f * defl);
      z -= dz;
      if (std::fabs(dz) < 1e-15) break;
    }
    x[1 + k] = z;
  }
  std::sort(x.begin(), x.end());
  return x;
}

// 1-D warp: equispaced -> Gauss-Lobatto displacement, equispaced Lagrange interpolant, over (1-xi^2)
struct Warp1D {
  int N;
  std::vector<double> xeq, disp;
  explicit Warp1D(int N_) : N(N_), xeq(N_ + 1), disp(N_ + 1) {
    const std::vector<double> gl = gauss_lobatto(N);
    for (int i = 0; i <= N; ++i) {
      xeq[i] = -1.0 + 2.0 * i / N;
      disp[i] = gl[i] - xeq[i];
    }
  }
  double operator()(double xi) const {
    if (std::fabs(xi) >= 1.0 - 1e-10) return 0.0;
    double w = 0.0;
    for (int i = 0; i <= N; ++i) {
      double l = 1.0;
      for (int j = 0; j <= N; ++j)
        if (j != i) l *= (xi - xeq[j]) / (xeq[i] - xeq[j]);
      w += disp[i] * l;
    }
    return w / (1.0 - xi * xi);
  }
};

// ---- dense helpers ---------------------------------------------------------------------------
// solve A X = B in place (A n x n row-major destroyed, B n x m row-major overwritten by X)
void lu_solve(std::vector<double> &A, std::vector<double> &B, int n, int m) {
  for (int c = 0; c < n; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r)
      if (std::fabs(A[(size_t)r * n + c]) > std::fabs(A[(size_t)piv * n + c])) piv = r;
    if (std::fabs(A[(size_t)piv * n + c]) < 1e-300) throw std::runtime_error("singular matrix in reference-element setup");
    if (piv != c) {
      for (int j = 0; j < n; ++j) std::swap(A[(size_t)c * n + j], A[(size_t)piv * n + j]);
      for (int j = 0; j < m; ++j) std::swap(B[(size_t)c * m + j], B[(size_t)piv * m + j]);
    }
    const double inv = 1.0 / A[(size_t)c * n + c];
    for (int r = c + 1; r < n; ++r) {
      const double f = A[(size_t)r * n + c] * inv;
      if (f == 0.0) continue;
      for (int j = c; j < n; ++j) A[(size_t)r * n + j] -= f * A[(size_t)c * n + j];
      for (int j = 0; j < m; ++j) B[(size_t)r * m + j] -= f * B[(size_t)c * m + j];
    }
  }
  for (int r = n - 1; r >= 0; --r) {
    for (int j = 0; j < m; ++j) {
      double acc = B[(size_t)r * m + j];
      for (int c = r + 1; c < n; ++c) acc -= A[(size_t)r * n + c] * B[(size_t)c * m + j];
      B[(size_t)r * m + j] = acc / A[(size_t)r * n + r];
    }
  }
}

// modal basis psi_ijk and its (r,s,t) gradient at one point
void dubiner3d(double r, double s, double t, int i, int j, int k, double &val, double &dr, double &ds, double &dt) {
  const double a = (std::fabs(s + t) > 1e-14) ? 2.0 * (1.0 + r) / (-s - t) - 1.0 : -1.0;
  const double b = (std::fabs(1.0 - t) > 1e-14) ? 2.0 * (1.0 + s) / (1.0 - t) - 1.0 : -1.0;
  const double c = t;
  const double fa = jac(i, 0.0, a), dfa = djac(i, 0.0, a);
  const double gb = jac(j, 2.0 * i + 1.0, b), dgb = djac(j, 2.0 * i + 1.0, b);
  const double hc = jac(k, 2.0 * (i + j) + 2.0, c), dhc = djac(k, 2.0 * (i + j) + 2.0, c);
  const double ob = 1.0 - b, oc = 1.0 - c;
  const double pb_i = std::pow(ob, i), pc_ij = std::pow(oc, i + j);
  const double pb_im1 = (i > 0) ? std::pow(ob, i - 1) : 0.0;
  const double pc_ijm1 = (i + j > 0) ? std::pow(oc, i + j - 1) : 0.0;
  const double sc = 2.0 * std::sqrt(2.0);
  val = sc * fa * gb * pb_i * hc * pc_ij;
  // d(gb (1-b)^i)/db and d(hc (1-c)^(i+j))/dc
  const double dB = dgb * pb_i - i * gb * pb_im1;
  const double dC = dhc * pc_ij - (i + j) * hc * pc_ijm1;
  // da/dr = 4/((1-b)(1-c)); da/ds = da/dt = 2(1+a)/((1-b)(1-c)); db/ds = 2/(1-c); db/dt = (1+b)/(1-c)
  const double core = dfa * gb * hc * pb_im1 * pc_ijm1;   // fa' B C / ((1-b)(1-c)), zero for i == 0
  const double mid = fa * dB * hc * pc_ijm1;              // fa B' C / (1-c), zero for i + j == 0
  dr = sc * 4.0 * core;
  ds = sc * (2.0 * (1.0 + a) * core + 2.0 * mid);
  dt = sc * (2.0 * (1.0 + a) * core + (1.0 + b) * mid + fa * gb * pb_i * dC);
}

double dubiner2d(double u, double w, int i, int j) {
  const double a = (std::fabs(1.0 - w) > 1e-14) ? 2.0 * (1.0 + u) / (1.0 - w) - 1.0 : -1.0;
  return std::sqrt(2.0) * jac(i, 0.0, a) * jac(j, 2.0 * i + 1.0, w) * std::pow(1.0 - w, i);
}

}  // namespace

// ================================================================================================
void build_refelem(int N, RefElem &ref) {
  if (N < 1 || N > 10) throw std::runtime_error("degree N must be in 1..10");
  const int Np = (N + 1) * (N + 2) * (N + 3) / 6, Nfp = (N + 1) * (N + 2) / 2;
  ref.N = N;
  ref.Np = Np;
  ref.Nfp = Nfp;
  // ---- warp-and-blend nodes (blend parameter 0, Q3)
  std::vector<double> lam((size_t)Np * 4);
  {
    int n = 0;
    for (int k = 0; k <= N; ++k)
      for (int j = 0; j <= N - k; ++j)
        for (int i = 0; i <= N - j - k; ++i, ++n) {
          lam[n * 4 + 1] = double(i) / N;
          lam[n * 4 + 2] = double(j) / N;
          lam[n * 4 + 3] = double(k) / N;
          lam[n * 4 + 0] = 1.0 - lam[n * 4 + 1] - lam[n * 4 + 2] - lam[n * 4 + 3];
        }
  }
  const double s3 = std::sqrt(3.0), s6 = std::sqrt(6.0);
  const double V[4][3] = {{-1.0, -1.0 / s3, -1.0 / s6}, {1.0, -1.0 / s3, -1.0 / s6}, {0.0, 2.0 / s3, -1.0 / s6}, {0.0, 0.0, 3.0 / s6}};
  const Warp1D warp(N);
  const double tol = 1e-10;
  ref.r.resize(Np);
  ref.s.resize(Np);
  ref.t.resize(Np);
  for (int n = 0; n < Np; ++n) {
    const double *L = &lam[n * 4];
    double X[3] = {0, 0, 0}, shift[3] = {0, 0, 0};
    for (int v = 0; v < 4; ++v)
      for (int d = 0; d < 3; ++d) X[d] += L[v] * V[v][d];
    for (int a = 0; a < 4; ++a) {  // face opposite vertex a
      int o[3], c = 0;
      for (int v = 0; v < 4; ++v)
        if (v != a) o[c++] = v;
      double W[3] = {0, 0, 0};
      for (int e = 0; e < 3; ++e) {  // edges o[e] -> o[e+1]
        const int u = o[e], v = o[(e + 1) % 3];
        double dir[3], len = 0.0;
        for (int d = 0; d < 3; ++d) {
          dir[d] = V[v][d] - V[u][d];
          len += dir[d] * dir[d];
        }
        len = std::sqrt(len);
        const double mag = 4.0 * L[u] * L[v] * warp(L[v] - L[u]);
        for (int d = 0; d < 3; ++d) W[d] += mag * dir[d] / len;
      }
      const double la = L[a], lb = L[o[0]], lc = L[o[1]], ld = L[o[2]];
      const double den = (lb + 0.5 * la) * (lc + 0.5 * la) * (ld + 0.5 * la);
      const double blend = (den > tol) ? lb * lc * ld / den : 0.0;
      for (int d = 0; d < 3; ++d) shift[d] += blend * W[d];
      const int inside = (lb > tol) + (lc > tol) + (ld > tol);
      if (la < tol && inside < 3)
        for (int d = 0; d < 3; ++d) shift[d] = W[d];
    }
    for (int d = 0; d < 3; ++d) X[d] += shift[d];
    // barycentric weights of the moved point w.r.t. the equilateral tetrahedron
    std::vector<double> A(9), rhs(3);
    for (int d = 0; d < 3; ++d) {
      for (int v = 0; v < 3; ++v) A[d * 3 + v] = V[v + 1][d] - V[0][d];
      rhs[d] = X[d] - V[0][d];
    }
    lu_solve(A, rhs, 3, 1);
    ref.r[n] = -1.0 + 2.0 * rhs[0];
    ref.s[n] = -1.0 + 2.0 * rhs[1];
    ref.t[n] = -1.0 + 2.0 * rhs[2];
  }
  // ---- Vandermonde and its gradients
  std::vector<double> Vm((size_t)Np * Np), Vr(Vm.size()), Vs(Vm.size()), Vt(Vm.size());
  {
    int col = 0;
    for (int i = 0; i <= N; ++i)
      for (int j = 0; j <= N - i; ++j)
        for (int k = 0; k <= N - i - j; ++k, ++col)
          for (int n = 0; n < Np; ++n)
            dubiner3d(ref.r[n], ref.s[n], ref.t[n], i, j, k, Vm[(size_t)n * Np + col], Vr[(size_t)n * Np + col],
                      Vs[(size_t)n * Np + col], Vt[(size_t)n * Np + col]);
  }
  // D = V_x V^-1: solve V^T D^T = V_x^T
  auto diffmat = [&](const std::vector<double> &Vx, std::vector<double> &D) {
    std::vector<double> At((size_t)Np * Np), Bt((size_t)Np * Np);
    for (int a = 0; a < Np; ++a)
      for (int b = 0; b < Np; ++b) {
        At[(size_t)a * Np + b] = Vm[(size_t)b * Np + a];
        Bt[(size_t)a * Np + b] = Vx[(size_t)b * Np + a];
      }
    lu_solve(At, Bt, Np, Np);
    D.resize((size_t)Np * Np);
    for (int a = 0; a < Np; ++a)
      for (int b = 0; b < Np; ++b) D[(size_t)a * Np + b] = Bt[(size_t)b * Np + a];
  };
  diffmat(Vr, ref.Dr);
  diffmat(Vs, ref.Ds);
  diffmat(Vt, ref.Dt);
  // ---- face masks
  ref.fmask.assign(4 * Nfp, -1);
  {
    int cnt[4] = {0, 0, 0, 0};
    for (int n = 0; n < Np; ++n) {
      const bool on[4] = {std::fabs(1.0 + ref.t[n]) < tol, std::fabs(1.0 + ref.s[n]) < tol,
                          std::fabs(1.0 + ref.r[n] + ref.s[n] + ref.t[n]) < tol, std::fabs(1.0 + ref.r[n]) < tol};
      for (int f = 0; f < 4; ++f)
        if (on[f]) {
          if (cnt[f] >= Nfp) throw std::runtime_error("reference element: too many nodes on a face");
          ref.fmask[f * Nfp + cnt[f]++] = n;
        }
    }
    for (int f = 0; f < 4; ++f)
      if (cnt[f] != Nfp) throw std::runtime_error("reference element: a face does not hold Nfp nodes");
  }
  // ---- merged lift matrix LIFT = V V^T E, E = face mass matrices (V_f V_f^T)^-1 scattered to face rows
  std::vector<double> E((size_t)Np * 4 * Nfp, 0.0);
  for (int f = 0; f < 4; ++f) {
    std::vector<double> Vf((size_t)Nfp * Nfp);
    for (int a = 0; a < Nfp; ++a) {
      const int n = ref.fmask[f * Nfp + a];
      const double u = (f <= 1) ? ref.r[n] : ref.s[n];
      const double w = (f == 0) ? ref.s[n] : ref.t[n];
      int col = 0;
      for (int i = 0; i <= N; ++i)
        for (int j = 0; j <= N - i; ++j, ++col) Vf[(size_t)a * Nfp + col] = dubiner2d(u, w, i, j);
    }
    std::vector<double> VVt((size_t)Nfp * Nfp, 0.0), Mf((size_t)Nfp * Nfp, 0.0);
    for (int a = 0; a < Nfp; ++a)
      for (int b = 0; b < Nfp; ++b) {
        double acc = 0.0;
        for (int c = 0; c < Nfp; ++c) acc += Vf[(size_t)a * Nfp + c] * Vf[(size_t)b * Nfp + c];
        VVt[(size_t)a * Nfp + b] = acc;
      }
    for (int a = 0; a < Nfp; ++a) Mf[(size_t)a * Nfp + a] = 1.0;
    lu_solve(VVt, Mf, Nfp, Nfp);
    for (int a = 0; a < Nfp; ++a)
      for (int b = 0; b < Nfp; ++b)
        E[(size_t)ref.fmask[f * Nfp + a] * 4 * Nfp + f * Nfp + b] = 0.5 * (Mf[(size_t)a * Nfp + b] + Mf[(size_t)b * Nfp + a]);
  }
  {
    const int nf = 4 * Nfp;
    std::vector<double> VtE((size_t)Np * nf, 0.0);
    for (int c = 0; c < Np; ++c)
      for (int n = 0; n < Np; ++n) {
        const double v = Vm[(size_t)n * Np + c];
        for (int j = 0; j < nf; ++j) VtE[(size_t)c * nf + j] += v * E[(size_t)n * nf + j];
      }
    ref.LIFT.assign((size_t)Np * nf, 0.0);
    for (int n = 0; n < Np; ++n)
      for (int c = 0; c < Np; ++c) {
        const double v = Vm[(size_t)n * Np + c];
        for (int j = 0; j < nf; ++j) ref.LIFT[(size_t)n * nf + j] += v * VtE[(size_t)c * nf + j];
      }
  }
  // ---- exterior-trace node table by barycentric matching on the reference faces
  ref.nbrnode.assign((size_t)4 * 4 * 6 * Nfp, 0xFFFF);
  ref.nbrface.assign((size_t)4 * 4 * 6 * Nfp, 0xFFFF);
  auto bary = [&](int n, int v) {
    switch (v) {
      case 0: return -(1.0 + ref.r[n] + ref.s[n] + ref.t[n]) / 2.0;
      case 1: return (1.0 + ref.r[n]) / 2.0;
      case 2: return (1.0 + ref.s[n]) / 2.0;
      default: return (1.0 + ref.t[n]) / 2.0;
    }
  };
  for (int f = 0; f < 4; ++f)
    for (int g = 0; g < 4; ++g)
      for (int s = 0; s < 6; ++s)
        for (int i = 0; i < Nfp; ++i) {
          const int n = ref.fmask[f * Nfp + i];
          int found = -1, found_ii = -1;
          for (int ii = 0; ii < Nfp; ++ii) {
            const int nn = ref.fmask[g * Nfp + ii];
            bool ok = true;
            for (int j = 0; j < 3 && ok; ++j)
              ok = std::fabs(bary(nn, FACE_VERTS[g][PERMS[s][j]]) - bary(n, FACE_VERTS[f][j])) < 1e-8;
            if (ok) {
              if (found >= 0) throw std::runtime_error("reference element: ambiguous face-node match");
              found = nn;
              found_ii = ii;
            }
          }
          if (found < 0) throw std::runtime_error("reference element: face node sets are not symmetric");
          ref.nbrnode[(((size_t)f * 4 + g) * 6 + s) * Nfp + i] = (uint16_t)found;
          ref.nbrface[(((size_t)f * 4 + g) * 6 + s) * Nfp + i] = (uint16_t)found_ii;
        }
}

// ================================================================================================
void build_mesh(int64_t nverts, int64_t K, const double *vxyz, const int32_t *etov, const int8_t *bc, HostMesh &m) {
  if (K <= 0 || nverts <= 0) throw std::runtime_error("mesh: empty mesh");
  if (K > (int64_t)0x1FFFFFFF) throw std::runtime_error("mesh: too many elements for 32-bit face indices");
  m.K = K;
  m.etov.assign(etov, etov + 4 * K);
  m.bctag.assign((size_t)4 * K, 1);
  if (bc) m.bctag.assign(bc, bc + 4 * K);
  m.verts.resize((size_t)K * 12);
  m.G.resize((size_t)K * 9);
  m.J.resize(K);
  m.nrm.resize((size_t)K * 12);
  m.fscale.resize((size_t)K * 4);
  for (int64_t k = 0; k < K; ++k) {
    int32_t *ev = &m.etov[4 * k];
    for (int v = 0; v < 4; ++v)
      if (ev[v] < 0 || ev[v] >= nverts) throw std::runtime_error("mesh: vertex index out of range");
    for (int pass = 0; pass < 2; ++pass) {
      const double *p[4];
      for (int v = 0; v < 4; ++v) p[v] = vxyz + 3 * (int64_t)ev[v];
      double A[3][3];  // columns x_r, x_s, x_t
      for (int d = 0; d < 3; ++d) {
        A[d][0] = 0.5 * (p[1][d] - p[0][d]);
        A[d][1] = 0.5 * (p[2][d] - p[0][d]);
        A[d][2] = 0.5 * (p[3][d] - p[0][d]);
      }
      const double det = A[0][0] * (A[1][1] * A[2][2] - A[1][2] * A[2][1]) - A[0][1] * (A[1][0] * A[2][2] - A[1][2] * A[2][0]) +
                         A[0][2] * (A[1][0] * A[2][1] - A[1][1] * A[2][0]);
      if (det < 0.0 && pass == 0) {  // fix orientation: swap the last two vertices (faces 0 and 1 trade places)
        std::swap(ev[2], ev[3]);
        std::swap(m.bctag[4 * k + 0], m.bctag[4 * k + 1]);
        continue;
      }
      double scale = 0.0;
      for (int d = 0; d < 3; ++d)
        for (int e = 0; e < 3; ++e) scale = std::max(scale, std::fabs(A[d][e]));
      if (!(det > 1e-14 * scale * scale * scale)) throw std::runtime_error("mesh: degenerate element (|J| ~ 0)");
      // inverse: rows are grad r, grad s, grad t
      double inv[3][3];
      inv[0][0] = (A[1][1] * A[2][2] - A[1][2] * A[2][1]) / det;
      inv[0][1] = (A[0][2] * A[2][1] - A[0][1] * A[2][2]) / det;
      inv[0][2] = (A[0][1] * A[1][2] - A[0][2] * A[1][1]) / det;
      inv[1][0] = (A[1][2] * A[2][0] - A[1][0] * A[2][2]) / det;
      inv[1][1] = (A[0][0] * A[2][2] - A[0][2] * A[2][0]) / det;
      inv[1][2] = (A[0][2] * A[1][0] - A[0][0] * A[1][2]) / det;
      inv[2][0] = (A[1][0] * A[2][1] - A[1][1] * A[2][0]) / det;
      inv[2][1] = (A[0][1] * A[2][0] - A[0][0] * A[2][1]) / det;
      inv[2][2] = (A[0][0] * A[1][1] - A[0][1] * A[1][0]) / det;
      m.J[k] = det;
      for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) m.G[9 * k + 3 * i + j] = inv[j][i];  // d r_j / d x_i
      for (int v = 0; v < 4; ++v)
        for (int d = 0; d < 3; ++d) m.verts[12 * k + 3 * v + d] = p[v][d];
      double nt[4][3];
      for (int d = 0; d < 3; ++d) {
        nt[0][d] = -inv[2][d];
        nt[1][d] = -inv[1][d];
        nt[2][d] = inv[0][d] + inv[1][d] + inv[2][d];
        nt[3][d] = -inv[0][d];
      }
      for (int f = 0; f < 4; ++f) {
        const double len = std::sqrt(nt[f][0] * nt[f][0] + nt[f][1] * nt[f][1] + nt[f][2] * nt[f][2]);
        m.fscale[4 * k + f] = len;
        for (int d = 0; d < 3; ++d) m.nrm[12 * k + 3 * f + d] = nt[f][d] / len;
      }
      break;
    }
  }
  // ---- face pairing: sort (sorted vertex triple, face id)
  struct FaceKey {
    int32_t a, b, c;
    uint32_t id;
  };
  std::vector<FaceKey> keys((size_t)4 * K);
  for (int64_t k = 0; k < K; ++k)
    for (int f = 0; f < 4; ++f) {
      int32_t v[3] = {m.etov[4 * k + FACE_VERTS[f][0]], m.etov[4 * k + FACE_VERTS[f][1]], m.etov[4 * k + FACE_VERTS[f][2]]};
      std::sort(v, v + 3);
      if (v[0] == v[1] || v[1] == v[2]) throw std::runtime_error("mesh: element with a repeated vertex");
      keys[4 * k + f] = {v[0], v[1], v[2], (uint32_t)(4 * k + f)};
    }
  std::sort(keys.begin(), keys.end(), [](const FaceKey &x, const FaceKey &y) {
    if (x.a != y.a) return x.a < y.a;
    if (x.b != y.b) return x.b < y.b;
    if (x.c != y.c) return x.c < y.c;
    return x.id < y.id;
  });
  m.nbr.assign((size_t)4 * K, -1);
  m.fcode.assign((size_t)4 * K, 255);
  auto same = [](const FaceKey &x, const FaceKey &y) { return x.a == y.a && x.b == y.b && x.c == y.c; };
  for (size_t i = 0; i < keys.size();) {
    size_t j = i + 1;
    while (j < keys.size() && same(keys[i], keys[j])) ++j;
    if (j - i > 2) throw std::runtime_error("mesh: non-conforming mesh (a face has more than two owners)");
    if (j - i == 2) {
      const uint32_t ids[2] = {keys[i].id, keys[i + 1].id};
      for (int side = 0; side < 2; ++side) {
        const int64_t k = ids[side] / 4, kk = ids[1 - side] / 4;
        const int f = ids[side] % 4, g = ids[1 - side] % 4;
        int code = -1;
        for (int s = 0; s < 6 && code < 0; ++s) {
          bool ok = true;
          for (int jv = 0; jv < 3 && ok; ++jv)
            ok = m.etov[4 * kk + FACE_VERTS[g][PERMS[s][jv]]] == m.etov[4 * k + FACE_VERTS[f][jv]];
          if (ok) code = s;
        }
        if (code < 0) throw std::runtime_error("mesh: internal error matching face vertices");
        m.nbr[4 * k + f] = (int32_t)kk;
        m.fcode[4 * k + f] = (uint8_t)(g * 6 + code);
        m.bctag[4 * k + f] = 0;
      }
    } else {
      const int64_t k = keys[i].id / 4;
      const int f = keys[i].id % 4;
      const int8_t tag = m.bctag[4 * k + f];
      if (tag < 1 || tag > 3) throw std::runtime_error("mesh: boundary face without a valid boundary tag");
    }
    i = j;
  }
}

}  // namespace dgh
