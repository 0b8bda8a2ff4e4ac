// Element partition and halo lists for the multi-GPU form of the hot path (host side).
//
// PAPER.md:22 ("weak element-to-element coupling"), PAPER.md:120 (data leave the GPU "for ... halo exchanges") and
// PAPER.md:475 (multi-GPU runs in the authors' ref. [33]): elements are independent within a stage except for the exterior
// traces of their faces.  One process per GPU owns a contiguous slab of the element list (for the cell-lexicographic Kuhn
// meshes of BASELINE.json: a slab of the cube) and keeps, behind its own elements, ghost copies of the elements on the
// other side of the cut faces.  Before every stage each rank sends, per peer, the face-node values (all fields) of its
// own elements on the cut faces -- Nfields x Nfp floats per cut face and direction -- and the peer stores them at the
// same volume nodes of its ghost copies, where the stage kernel's gather finds them like any other neighbour.
//
// This file builds the local mesh of one rank and the send / receive lists; dg_api.cu has the device pack / unpack
// kernels (dg_halo_pack / dg_halo_unpack) and the `owned_elements` option that keeps the stage kernels off the ghosts.
#include <algorithm>
#include <cstring>
#include <map>
#include <new>
#include <stdexcept>
#include <string>
#include <vector>

#include "../../include/dg.h"
#include "host_setup.hpp"

struct dg_part {
  int nranks = 1, rank = 0;
  int64_t K = 0, k0 = 0, k1 = 0;                 // global size, owned range [k0, k1)
  std::vector<int64_t> ghosts;                   // global ids, ascending (hence grouped by owner)
  std::vector<int32_t> etov;                     // [owned + ghost][4], caller's vertex order, global vertex numbers
  std::vector<int8_t> bc;                        // [owned + ghost][4], caller's face numbering
  struct Peer {
    int rank;
    std::vector<int32_t> send, recv;             // 4 * local element + face (library face numbering), ordered by (global element, face)
  };
  std::vector<Peer> peers;
};

namespace dgapi {
int fail(int code, const std::string &msg);       // dg_api.cu: sets the thread-local message
}

namespace {
int64_t slab_begin(int64_t K, int nranks, int r) { return K * r / nranks; }
int owner_of(int64_t K, int nranks, int64_t k) {
  int r = (int)((k * nranks) / K);
  while (r > 0 && slab_begin(K, nranks, r) > k) --r;
  while (r + 1 < nranks && slab_begin(K, nranks, r + 1) <= k) ++r;
  return r;
}
}  // namespace

extern "C" {

int dg_partition_create(dg_part **out, const dg_mesh *mesh, int nranks, int rank) {
  if (!out) return dgapi::fail(DG_ERR_ARG, "out is NULL");
  *out = nullptr;
  if (!mesh || !mesh->vxyz || !mesh->etov) return dgapi::fail(DG_ERR_ARG, "NULL input pointer");
  if (nranks < 1 || rank < 0 || rank >= nranks) return dgapi::fail(DG_ERR_ARG, "need 0 <= rank < nranks");
  if (mesh->K < nranks) return dgapi::fail(DG_ERR_MESH, "mesh: fewer elements than ranks");
  dg_part *p = new (std::nothrow) dg_part();
  if (!p) return dgapi::fail(DG_ERR_NOMEM, "out of host memory");
  try {
    dgh::HostMesh m;                              // global connectivity (library orientation and face numbering)
    dgh::build_mesh(mesh->nverts, mesh->K, mesh->vxyz, mesh->etov, mesh->bc, m);
    const int64_t K = mesh->K;
    p->nranks = nranks; p->rank = rank; p->K = K;
    p->k0 = slab_begin(K, nranks, rank);
    p->k1 = slab_begin(K, nranks, rank + 1);
    // ghosts = elements of other ranks across a face of an owned element
    for (int64_t k = p->k0; k < p->k1; ++k)
      for (int f = 0; f < 4; ++f) {
        const int64_t nb = m.nbr[4 * k + f];
        if (nb >= 0 && (nb < p->k0 || nb >= p->k1)) p->ghosts.push_back(nb);
      }
    std::sort(p->ghosts.begin(), p->ghosts.end());
    p->ghosts.erase(std::unique(p->ghosts.begin(), p->ghosts.end()), p->ghosts.end());
    const int64_t nown = p->k1 - p->k0, ngh = (int64_t)p->ghosts.size();
    auto local_of = [&](int64_t g) -> int64_t {
      if (g >= p->k0 && g < p->k1) return g - p->k0;
      auto it = std::lower_bound(p->ghosts.begin(), p->ghosts.end(), g);
      if (it == p->ghosts.end() || *it != g) throw std::runtime_error("mesh: internal error (element is neither owned nor ghost)");
      return nown + (it - p->ghosts.begin());
    };
    // local mesh rows: the caller's own rows (dg_create will orient them exactly as it did here)
    p->etov.resize((size_t)(nown + ngh) * 4);
    p->bc.assign((size_t)(nown + ngh) * 4, (int8_t)DG_BC_RIGID);
    for (int64_t l = 0; l < nown + ngh; ++l) {
      const int64_t g = l < nown ? p->k0 + l : p->ghosts[l - nown];
      std::memcpy(&p->etov[4 * l], mesh->etov + 4 * g, 4 * sizeof(int32_t));
      // owned elements keep the caller's tags; a ghost's faces towards elements that are not here are never evaluated
      // (ghosts are not advanced): they only need some valid tag
      if (l < nown && mesh->bc) std::memcpy(&p->bc[4 * l], mesh->bc + 4 * g, 4);
    }
    // halo lists per peer
    std::map<int, dg_part::Peer> peers;
    struct Ent { int64_t g; int f; };
    std::map<int, std::vector<Ent>> send, recv;
    for (int64_t k = p->k0; k < p->k1; ++k)
      for (int f = 0; f < 4; ++f) {
        const int64_t nb = m.nbr[4 * k + f];
        if (nb < 0 || (nb >= p->k0 && nb < p->k1)) continue;
        const int r = owner_of(K, nranks, nb);
        send[r].push_back({k, f});                               // my element's trace on the cut face
        recv[r].push_back({nb, (int)(m.fcode[4 * k + f] / 6)});  // the neighbour's trace on its side of the same face
      }
    for (auto &kv : send) {
      dg_part::Peer pr;
      pr.rank = kv.first;
      auto cmp = [](const Ent &a, const Ent &b) { return a.g != b.g ? a.g < b.g : a.f < b.f; };
      std::sort(kv.second.begin(), kv.second.end(), cmp);
      auto &rv = recv[kv.first];
      std::sort(rv.begin(), rv.end(), cmp);
      for (const Ent &e : kv.second) pr.send.push_back((int32_t)(4 * local_of(e.g) + e.f));
      for (const Ent &e : rv) pr.recv.push_back((int32_t)(4 * local_of(e.g) + e.f));
      p->peers.push_back(std::move(pr));
    }
  } catch (const std::bad_alloc &) {
    delete p;
    return dgapi::fail(DG_ERR_NOMEM, "out of host memory");
  } catch (const std::exception &e) {
    delete p;
    const std::string msg = e.what();
    return dgapi::fail(msg.rfind("mesh:", 0) == 0 ? DG_ERR_MESH : DG_ERR_ARG, msg);
  }
  *out = p;
  return DG_OK;
}

int dg_partition_destroy(dg_part *p) {
  if (!p) return dgapi::fail(DG_ERR_ARG, "NULL partition");
  delete p;
  return DG_OK;
}

int64_t dg_partition_num_owned(const dg_part *p) { return p ? p->k1 - p->k0 : (int64_t)dgapi::fail(DG_ERR_ARG, "NULL partition"); }
int64_t dg_partition_num_ghost(const dg_part *p) { return p ? (int64_t)p->ghosts.size() : (int64_t)dgapi::fail(DG_ERR_ARG, "NULL partition"); }

int dg_partition_global_ids(const dg_part *p, int64_t *ids) {
  if (!p || !ids) return dgapi::fail(DG_ERR_ARG, "NULL argument");
  const int64_t nown = p->k1 - p->k0;
  for (int64_t l = 0; l < nown; ++l) ids[l] = p->k0 + l;
  std::copy(p->ghosts.begin(), p->ghosts.end(), ids + nown);
  return DG_OK;
}

int dg_partition_local_mesh(const dg_part *p, int32_t *etov, int8_t *bc) {
  if (!p) return dgapi::fail(DG_ERR_ARG, "NULL partition");
  if (etov) std::memcpy(etov, p->etov.data(), p->etov.size() * sizeof(int32_t));
  if (bc) std::memcpy(bc, p->bc.data(), p->bc.size());
  return DG_OK;
}

int dg_partition_num_peers(const dg_part *p) { return p ? (int)p->peers.size() : dgapi::fail(DG_ERR_ARG, "NULL partition"); }

int dg_partition_peer(const dg_part *p, int i, int *rank, int64_t *nsend, int64_t *nrecv) {
  if (!p || i < 0 || i >= (int)p->peers.size()) return dgapi::fail(DG_ERR_ARG, "bad peer index");
  if (rank) *rank = p->peers[i].rank;
  if (nsend) *nsend = (int64_t)p->peers[i].send.size();
  if (nrecv) *nrecv = (int64_t)p->peers[i].recv.size();
  return DG_OK;
}

int dg_partition_halo_faces(const dg_part *p, int i, int32_t *send_faces, int32_t *recv_faces) {
  if (!p || i < 0 || i >= (int)p->peers.size()) return dgapi::fail(DG_ERR_ARG, "bad peer index");
  const dg_part::Peer &pr = p->peers[i];
  if (send_faces) std::memcpy(send_faces, pr.send.data(), pr.send.size() * sizeof(int32_t));
  if (recv_faces) std::memcpy(recv_faces, pr.recv.data(), pr.recv.size() * sizeof(int32_t));
  return DG_OK;
}

}  // extern "C"
