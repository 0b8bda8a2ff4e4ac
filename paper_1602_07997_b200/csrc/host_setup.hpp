// Host-side setup of libdg: reference-element operators, geometric factors, connectivity.
// fp64 throughout; rounded once to fp32 when uploaded.  Independent of oracle/ (shares no code).
// Conventions: include/dg.h; definitions the paper defers to its ref [33] follow
// DESIGN.md readings Q3 (nodes), Q4 (operators), Q5 (g^vol index order).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

namespace dgh {

struct RefElem {
  int N = 0, Np = 0, Nfp = 0;
  std::vector<double> r, s, t;          // nodes, lattice order (t slowest, r fastest)
  std::vector<double> Dr, Ds, Dt;       // [Np][Np] row-major
  std::vector<double> LIFT;             // [Np][4Nfp] row-major, merged lift matrix
  std::vector<int32_t> fmask;           // [4][Nfp] volume node of each face node
  // exterior-trace node table: for my face f, neighbour face g, vertex correspondence s (0..5):
  // nbrnode[((f*4+g)*6+s)*Nfp + i] = volume node (in the neighbour) that coincides with my face node i
  std::vector<uint16_t> nbrnode;
  std::vector<uint16_t> nbrface;        // same indexing: that node's position i' on the neighbour's face g (fmask[g][i'] = nbrnode[...])
};

// the six correspondences: neighbour face-local vertex PERMS[s][j] coincides with my face-local vertex j
extern const int PERMS[6][3];
extern const int FACE_VERTS[4][3];

void build_refelem(int N, RefElem &ref);      // throws std::runtime_error

struct HostMesh {
  int64_t K = 0;
  std::vector<int32_t> etov;            // [K][4] after orientation fix
  std::vector<int8_t> bctag;            // [K][4] 0 interior else DG_BC_*
  std::vector<double> verts;            // [K][4][3] vertex coordinates per element
  std::vector<double> G;                // [K][3][3], G[i][j] = d r_j / d x_i
  std::vector<double> J;                // [K]
  std::vector<double> nrm;              // [K][4][3]
  std::vector<double> fscale;           // [K][4]  sJ/J
  std::vector<int32_t> nbr;             // [K][4] neighbour element, -1 on the boundary
  std::vector<uint8_t> fcode;           // [K][4] g*6+s for interior faces, 255 on the boundary
};

// throws std::runtime_error with a message starting "mesh:" on bad input
void build_mesh(int64_t nverts, int64_t K, const double *vxyz, const int32_t *etov, const int8_t *bc,
                HostMesh &m);

}  // namespace dgh
