// libdg C ABI (include/dg.h): context, host setup -> device upload, kernel dispatch.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <array>
#include <new>
#include <stdexcept>
#include <string>
#include <vector>

#include "../../include/dg.h"
#include "dg_prof.h"
#include "host_setup.hpp"
#include "kernels.cuh"
#include "tc3_kernels.cuh"
#include "iface_kernels.cuh"

// per-(model, degree) kernel getters from stage_inst.cu
#define DG_DECL(m, n)                                              \
  extern "C" const void *dgk_get_stage_kernel_##m##_##n(int, int); \
  extern "C" size_t dgk_stage_smem_bytes_##m##_##n(int);           \
  extern "C" const void *dgk_get_tc3_kernel_##m##_##n(int);       \
  extern "C" const void *dgk_get_epk_kernel_##m##_##n(int);       \
  extern "C" int dgk_epk_upload_##m##_##n(const float *, const float *, const unsigned short *, const int *); \
  extern "C" const void *dgk_get_iface_kernel_##m##_##n(void);   \
  extern "C" int dgk_tc3_info_##m##_##n(int);                     \
  extern "C" const void *dgk_get_rpt_kernel_##m##_##n(int);       \
  extern "C" int dgk_rpt_info_##m##_##n(int);                     \
  extern "C" int dgk_rpt_upload_##m##_##n(const float *, const float *);
#define DG_DECL_ALL(m) \
  DG_DECL(m, 1) DG_DECL(m, 2) DG_DECL(m, 3) DG_DECL(m, 4) DG_DECL(m, 5) DG_DECL(m, 6) DG_DECL(m, 7) DG_DECL(m, 8) DG_DECL(m, 9) DG_DECL(m, 10)
DG_DECL_ALL(0)
DG_DECL_ALL(1)

#ifdef DG_PROF
#define DG_DECLP(m, n) extern "C" int dgk_prof_read_##m##_##n(long long *);
#define DG_DECLP_ALL(m) DG_DECLP(m, 1) DG_DECLP(m, 2) DG_DECLP(m, 3) DG_DECLP(m, 4) DG_DECLP(m, 5) DG_DECLP(m, 6) DG_DECLP(m, 7) DG_DECLP(m, 8) DG_DECLP(m, 9) DG_DECLP(m, 10)
DG_DECLP_ALL(0)
DG_DECLP_ALL(1)
#endif

namespace {
typedef const void *(*kernel_getter)(int, int);
typedef size_t (*smem_getter)(int);
typedef const void *(*tc_getter)(int);
typedef int (*info_getter)(int);
#define DG_ROW(m, fn)                                                                                          \
  {nullptr, fn##m##_1, fn##m##_2, fn##m##_3, fn##m##_4, fn##m##_5, fn##m##_6, fn##m##_7, fn##m##_8, fn##m##_9, \
   fn##m##_10}
const kernel_getter KERNELS[2][11] = {DG_ROW(0, dgk_get_stage_kernel_), DG_ROW(1, dgk_get_stage_kernel_)};
const smem_getter SMEM[2][11] = {DG_ROW(0, dgk_stage_smem_bytes_), DG_ROW(1, dgk_stage_smem_bytes_)};
typedef int (*epk_upload_fn)(const float *, const float *, const unsigned short *, const int *);
const tc_getter EPK_KERNELS[2][11] = {DG_ROW(0, dgk_get_epk_kernel_), DG_ROW(1, dgk_get_epk_kernel_)};
const epk_upload_fn EPK_UPLOAD[2][11] = {DG_ROW(0, dgk_epk_upload_), DG_ROW(1, dgk_epk_upload_)};
const tc_getter TC3_KERNELS[2][11] = {DG_ROW(0, dgk_get_tc3_kernel_), DG_ROW(1, dgk_get_tc3_kernel_)};
const info_getter TC3_INFO[2][11] = {DG_ROW(0, dgk_tc3_info_), DG_ROW(1, dgk_tc3_info_)};
typedef int (*rpt_upload_fn)(const float *, const float *);
const tc_getter RPT_KERNELS[2][11] = {DG_ROW(0, dgk_get_rpt_kernel_), DG_ROW(1, dgk_get_rpt_kernel_)};
const info_getter RPT_INFO[2][11] = {DG_ROW(0, dgk_rpt_info_), DG_ROW(1, dgk_rpt_info_)};
const rpt_upload_fn RPT_UPLOAD[2][11] = {DG_ROW(0, dgk_rpt_upload_), DG_ROW(1, dgk_rpt_upload_)};
typedef const void *(*iface_getter)(void);
const iface_getter IFACE_KERNELS[2][11] = {DG_ROW(0, dgk_get_iface_kernel_), DG_ROW(1, dgk_get_iface_kernel_)};

thread_local std::string g_err;
int fail(int code, const std::string &msg) {
  g_err = msg;
  return code;
}
}  // namespace
namespace dgapi {
int fail(int code, const std::string &msg) { return ::fail(code, msg); }
}  // namespace dgapi
namespace {
#define CUDA_TRY(x)                                                                                   \
  do {                                                                                                \
    cudaError_t e_ = (x);                                                                             \
    if (e_ != cudaSuccess) throw std::runtime_error(std::string("cuda: ") + cudaGetErrorString(e_) + " at " #x); \
  } while (0)

// LSRK(5,4) of Carpenter & Kennedy (BASELINE.json north_star; Q2), exact rationals
const double RK_A[5] = {0.0, -567301805773.0 / 1357537059087.0, -2404267990393.0 / 2016746695238.0,
                        -3550918686646.0 / 2091501179385.0, -1275806237668.0 / 842570457699.0};
const double RK_B[5] = {1432997174477.0 / 9575080441755.0, 5161836677717.0 / 13612068292357.0,
                        1720146321549.0 / 2090206949498.0, 3134564353537.0 / 4481467310338.0,
                        2277821191437.0 / 14882151754819.0};
}  // namespace

namespace dgk {
// rows of `np` floats from pitch `spitch` to pitch `dpitch` (caller layout <-> the tensor-core kernel's padded rows)
__global__ void repitch_kernel(float *__restrict__ dst, int dpitch, const float *__restrict__ src, int spitch, int np, size_t n) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t r = i / (unsigned)np;
    const int c = (int)(i - r * (unsigned)np);
    dst[r * dpitch + c] = src[r * spitch + c];
  }
}

// halo exchange (partition.cpp): face-node values of all fields of the listed faces (4 element + face) <-> a dense buffer
// [face][field][face node]; the same routine on the sending side (pack, owned elements) and the receiving side (unpack, ghosts)
template <bool PACK>
__global__ void halo_kernel(float *__restrict__ q, float *__restrict__ buf, const int *__restrict__ faces, const unsigned short *__restrict__ fmask,
                            int nf, int np, int nfp, size_t n) {
  for (size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += (size_t)gridDim.x * blockDim.x) {
    const size_t ent = t / (unsigned)(nf * nfp);
    const int rem = (int)(t - ent * (unsigned)(nf * nfp));
    const int c = rem / nfp, i = rem - c * nfp;
    const int fa = faces[ent];
    float *qq = q + ((size_t)(fa >> 2) * nf + c) * np + fmask[(fa & 3) * nfp + i];
    if (PACK) buf[t] = *qq;
    else *qq = buf[t];
  }
}

}  // namespace dgk

struct dg_ctx {
  int N = 0, Np = 0, Nfp = 0, model = 0, NF = 0, device = -1;
  int64_t K = 0;
  int64_t K_active = 0;                          // elements the stage kernels advance (dg_options.owned_elements; the rest are ghosts)
  dgh::RefElem ref;
  dgh::HostMesh mesh;
  std::vector<double> cmax;
  // device constants and scratch
  float *d_DT = nullptr, *d_LT = nullptr, *d_geo = nullptr;
  int *d_nbr = nullptr;
  unsigned char *d_fcode = nullptr;
  unsigned short *d_fmask = nullptr, *d_nbrnode = nullptr;
  uint16_t *d_Bimg = nullptr;                    // tensor-core variant: bf16x3 operator panel image
  bool tc3 = false;                              // pipelined BF16x3 tensor-core variant (tc3_kernels.cuh)
  bool rpt = false;                              // row-per-thread kernel (rpt_kernels.cuh): N <= 3
  int rpt_epc = 0;                               // its elements per CTA and tile round
  int rpt_cap = 0;                               // its persistent grid: resident CTAs per SM x SMs (set at the first launch)
  bool epk = false;                              // element-per-thread kernel (epk_kernels.cuh): acoustic N <= 2, elastic N = 1
  int *d_conn = nullptr;                         // tc3: packed connectivity [K][4]
  int epi_cw = 0;                                // tc3: epilogue chunk width (TMA box columns)
  int PT = 0;                                    // tc3: row pitch (floats) of the arrays the kernel works on, Np rounded up to 4
  float *d_qa = nullptr;                         // tc3, PT != Np: padded private copies of the state (d_qa and d_q2 ping-pong)
  // device array -> TMA descriptors (epilogue boxes of height 32 / Nf EB - 96; field chunks).  Library-owned buffers are
  // encoded at dg_create and pinned; caller buffers are encoded on first sight (host-side work only, no device
  // allocation) and the oldest unpinned entry is evicted beyond TMAP_CACHE entries
  struct TmapEntry { std::array<CUtensorMap, 5> m; bool pinned; uint64_t stamp; };
  std::map<const void *, TmapEntry> tmaps;
  uint64_t tmap_clock = 0;
  // interface-centric surface step (dg_options.surface = 1, iface_kernels.cuh)
  int surface = 0;
  const void *k_iface = nullptr;
  float *d_pflux = nullptr;                      // [K][Nf][4 Nfp] penalty terms times g^sur
  int *d_ifaces = nullptr;                       // interior owner faces, then boundary faces
  unsigned short *d_nbrface = nullptr;
  int n_int = 0, n_bnd = 0;
  int iface_launches = 0;                        // interface kernels launched by the current API call
  int max_ctas = 0;                              // dg_options.max_ctas: cap on the persistent grid (tests; 0 = one CTA per SM)
  float *d_res = nullptr, *d_q2 = nullptr, *d_hist[3] = {nullptr, nullptr, nullptr};
  int hist_head = 0;                             // d_hist[hist_head] = r^{m-1}, d_hist[(hist_head + 1) % 3] = r^{m-2}
  int nhist = 0;                                 // AB3: right-hand sides of earlier steps on record (start-up while < 2)
  // launch configuration
  const void *k_rhs = nullptr, *k_stage = nullptr, *k_ab3 = nullptr;
  int E = 0, G = 0, NT = 0, grid = 0;
  size_t smem = 0;
  int nbatch = 0, num_sms = 0;
  int last_launches = 0;
  std::string variant;
};

// ---- work memory of dg_step_static (include/dg.h): a file-scope device array instead of cudaMalloc'ed buffers, for callers
// that must not allocate.  Every GPU that loads the library holds these DG_STATIC_SCRATCH_BYTES until the process exits.
// In host code the name is only a stand-in: the device address comes from cudaGetSymbolAddress (static_scratch_setup),
// once per device, with that device current.
static __device__ __align__(256) unsigned char dg_static_scratch[DG_STATIC_SCRATCH_BYTES];

namespace {

// Every device entry point runs on the context's device and leaves the caller's current device as it found it.
struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    if (prev != dev) ok = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceGuard() {
    int cur = -1;
    if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
  }
};
constexpr int STATIC_SCRATCH_MAX_DEVICES = 64;
std::mutex g_scratch_mu;
unsigned char *g_scratch_ptr[STATIC_SCRATCH_MAX_DEVICES];      // device address of dg_static_scratch, per device
int g_scratch_state[STATIC_SCRATCH_MAX_DEVICES];               // 0 = not asked yet, 1 = resolved, else -(cudaError_t)
// Resolves the device address of dg_static_scratch on device `dev`, which must be current (dg_create and dg_step_static hold
// a DeviceGuard).  Called at set-up by dg_create; never fatal there: a failure is kept and reported by dg_step_static.
void static_scratch_setup(int dev) {
  if (dev < 0 || dev >= STATIC_SCRATCH_MAX_DEVICES) return;
  std::lock_guard<std::mutex> lock(g_scratch_mu);
  if (g_scratch_state[dev] == 1) return;
  void *ptr = nullptr;
  const cudaError_t e = cudaGetSymbolAddress(&ptr, dg_static_scratch);
  if (e == cudaSuccess && ptr) {
    g_scratch_ptr[dev] = static_cast<unsigned char *>(ptr);
    g_scratch_state[dev] = 1;
  } else {
    g_scratch_state[dev] = e == cudaSuccess ? -(int)cudaErrorInvalidSymbol : -(int)e;
    (void)cudaGetLastError();
  }
}

template <class T>
T *upload(const std::vector<T> &h) {
  T *d = nullptr;
  CUDA_TRY(cudaMalloc(&d, std::max<size_t>(h.size(), 1) * sizeof(T)));
  CUDA_TRY(cudaMemcpy(d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
  return d;
}

void free_device(dg_ctx *c) {
  if (c->device < 0) return;
  DeviceGuard guard(c->device);
  cudaFree(c->d_DT); cudaFree(c->d_LT); cudaFree(c->d_Bimg); cudaFree(c->d_conn); cudaFree(c->d_qa); cudaFree(c->d_geo); cudaFree(c->d_nbr); cudaFree(c->d_fcode);
  cudaFree(c->d_fmask); cudaFree(c->d_nbrnode); cudaFree(c->d_res); cudaFree(c->d_q2);
  for (float *&h : c->d_hist) cudaFree(h);
  cudaFree(c->d_pflux); cudaFree(c->d_ifaces); cudaFree(c->d_nbrface);
}

void build_geo_records(const dg_ctx *c, const dg_materials *mat, std::vector<float> &geo) {
  const int64_t K = c->K;
  const int NG = c->model == DG_ACOUSTIC ? dgk::GEO_AC : dgk::GEO_EL;
  geo.assign((size_t)K * NG, 0.f);
  const dgh::HostMesh &m = c->mesh;
  for (int64_t k = 0; k < K; ++k) {
    float *g = &geo[(size_t)k * NG];
    for (int i = 0; i < 9; ++i) g[i] = (float)m.G[9 * k + i];
    const double rho = mat->rho[k], cp = mat->c_or_vp[k];
    if (c->model == DG_ACOUSTIC) {
      g[9] = (float)(rho * cp * cp);
      g[10] = (float)(1.0 / rho);
      g[11] = (float)cp;
      const double Zm = rho * cp;
      for (int f = 0; f < 4; ++f) {
        const int64_t kk = m.nbr[4 * k + f] >= 0 ? m.nbr[4 * k + f] : k;
        const double Zp = mat->rho[kk] * mat->c_or_vp[kk];
        float *fg = g + 12 + 5 * f;
        for (int d = 0; d < 3; ++d) fg[d] = (float)m.nrm[12 * k + 3 * f + d];
        fg[3] = (float)(m.fscale[4 * k + f] / (Zm + Zp));   // g^sur k_c / 2, k_c = 1/{rho c}
        fg[4] = (float)Zp;
      }
    } else {
      const double cs = mat->vs[k];
      const double mu = rho * cs * cs, lam = rho * cp * cp - 2.0 * mu;
      g[9] = (float)(1.0 / rho);
      g[10] = (float)lam;
      g[11] = (float)mu;
      g[12] = (float)cp;
      g[13] = (float)cs;
      for (int f = 0; f < 4; ++f) {
        const int64_t kk = m.nbr[4 * k + f] >= 0 ? m.nbr[4 * k + f] : k;
        const double Zpp = mat->rho[kk] * mat->c_or_vp[kk], Zsp = mat->rho[kk] * mat->vs[kk];
        float *fg = g + 16 + 8 * f;
        for (int d = 0; d < 3; ++d) fg[d] = (float)m.nrm[12 * k + 3 * f + d];
        fg[3] = (float)(m.fscale[4 * k + f] / (rho * cp + Zpp));
        fg[4] = (float)(m.fscale[4 * k + f] / (rho * cs + Zsp));
        fg[5] = (float)Zpp;
        fg[6] = (float)Zsp;
      }
    }
  }
}

// round to nearest even bf16; returns the 16-bit pattern and the value
uint16_t bf16_rn(double x, double &val) {
  float f = (float)x;
  uint32_t u;
  std::memcpy(&u, &f, 4);
  u = (u + 0x7FFFu + ((u >> 16) & 1u)) & 0xFFFF0000u;
  std::memcpy(&f, &u, 4);
  val = (double)f;
  return (uint16_t)(u >> 16);
}

// Operator panel of the tensor-core variant as the shared-memory image of every k-step (tc3_kernels.cuh): the output
// nodes are split into NSPLIT contiguous ranges of NCH rows, one image per range:
// [half][step][piece 3][kc 2][NCH rows n][8 k] bf16, K-major core matrices of 8 rows x 16 bytes.  Step 3g + j holds
// D_j[n][16g + k], step 3 NG + h holds LIFT[n][16h + k]; entries beyond Np / 4Nfp are zero.  Pieces: BF16x3 split of
// the fp64 operator entry, b1 = bf16(x), b2 = bf16(x - b1), b3 = bf16(x - b1 - b2).
void build_tc3_image(const dgh::RefElem &ref, int NCH, int nsplit, int nstep, std::vector<uint16_t> &img) {
  const int Np = ref.Np, NFACE = 4 * ref.Nfp;
  const int NG = (Np + 15) / 16;
  const size_t stage = (size_t)3 * 2 * NCH * 8;
  img.assign((size_t)nsplit * nstep * stage, 0);
  const std::vector<double> *Dm[3] = {&ref.Dr, &ref.Ds, &ref.Dt};
  auto put = [&](int st, int n, int k, double v) {
    double v1, v2, v3;
    const uint16_t b1 = bf16_rn(v, v1), b2 = bf16_rn(v - v1, v2), b3 = bf16_rn(v - v1 - v2, v3);
    const int half = n / NCH, nn = n - half * NCH;
    const size_t off = ((size_t)half * nstep + st) * stage + (size_t)(k >> 3) * NCH * 8 + (size_t)nn * 8 + (k & 7);
    img[off] = b1;
    img[off + (size_t)2 * NCH * 8] = b2;
    img[off + (size_t)4 * NCH * 8] = b3;
  };
  for (int g = 0; g < NG; ++g)
    for (int j = 0; j < 3; ++j)
      for (int k = 0; k < 16; ++k) {
        const int m = 16 * g + k;
        if (m >= Np) continue;
        for (int n = 0; n < Np; ++n) put(3 * g + j, n, k, (*Dm[j])[(size_t)n * Np + m]);
      }
  for (int st = 3 * NG; st < nstep; ++st)
    for (int k = 0; k < 16; ++k) {
      const int jf = 16 * (st - 3 * NG) + k;
      if (jf >= NFACE) continue;
      for (int n = 0; n < Np; ++n) put(st, n, k, ref.LIFT[(size_t)n * NFACE + jf]);
    }
}

void choose_variant(dg_ctx *c, const dg_options *o) {
  int want = o ? o->variant : 0;
  // auto (config-4 sweep): the tensor-core kernel from N = 3 up; the row-per-thread kernel at N = 2
  // (acoustic 0.74 vs 0.79 ms element per thread; elastic 1.98 vs 2.62 ms tensor core); the element-per-thread kernel at N = 1
  // (Np = 4: three of four k-steps of the tensor-core kernel would be padding) -- an explicit launch shape asks for the
  // fused node-per-thread kernel
  if (want == 0) {
    const bool shape = o && (o->elems_per_thread > 0 || o->groups_per_cta > 0);
    want = shape ? 1 : ((c->N >= 3 && c->K < (1 << 26)) ? 4 : (c->N == 2 ? 5 : 1));
  }
  if (want != 1 && want != 4 && want != 5)
    throw std::invalid_argument("unknown variant (0 auto, 1 fused FP32 SIMT, 4 pipelined tensor core BF16x3, 5 FP32 SIMT row per thread)");
  if (want == 5) {
    if (!RPT_KERNELS[c->model][c->N](dgk::MODE_STAGE)) throw std::invalid_argument("the row-per-thread variant covers N <= 3");
    c->rpt = true;
    c->k_rhs = RPT_KERNELS[c->model][c->N](dgk::MODE_RHS);
    c->k_stage = RPT_KERNELS[c->model][c->N](dgk::MODE_STAGE);
    c->k_ab3 = RPT_KERNELS[c->model][c->N](dgk::MODE_AB3);
    c->NT = RPT_INFO[c->model][c->N](0);
    c->rpt_epc = RPT_INFO[c->model][c->N](1);
    c->smem = 0;
    c->grid = (int)((c->K_active + c->rpt_epc - 1) / c->rpt_epc);
    char buf[160];
    snprintf(buf, sizeof buf, "simt_row_per_thread<%s,N=%d,threads=%d,elems/cta=%d,operators in constant memory>",
             c->model == DG_ACOUSTIC ? "acoustic" : "elastic", c->N, c->NT, c->rpt_epc);
    c->variant = buf;
    return;
  }
  if (want == 4) {
    if (c->K >= (1 << 26)) throw std::invalid_argument("pipelined tensor-core variant packs the neighbour in 26 bits: K < 2^26");
    c->tc3 = true;
    c->k_rhs = TC3_KERNELS[c->model][c->N](dgk::MODE_RHS);
    c->k_stage = TC3_KERNELS[c->model][c->N](dgk::MODE_STAGE);
    c->k_ab3 = TC3_KERNELS[c->model][c->N](dgk::MODE_AB3);
    const info_getter info = TC3_INFO[c->model][c->N];
    const int EB = info(1);
    c->nbatch = (int)((c->K_active + EB - 1) / EB);
    c->NT = dgk::T3_THREADS;
    c->smem = (size_t)info(0);
    c->epi_cw = info(9);
    c->PT = info(10);
    char buf[240];
    snprintf(buf, sizeof buf, "tc_pipe_bf16x3<%s,N=%d,NCH=%d,nsplit=%d,elems/batch=%d,ksteps=%d,tile=%s x%d,accsets=%d,aring=%d,pitch=%d,threads=%d,smem=%zu>",
             c->model == DG_ACOUSTIC ? "acoustic" : "elastic", c->N, info(2), info(4), EB, info(3), info(5) ? "smem" : "L1", info(6), info(7),
             info(8), info(10), c->NT, c->smem);
    c->variant = buf;
    return;
  }
  const int Np = c->Np;
  // lowest degrees: one element per thread, everything in registers -- unless a launch shape of the generic kernel is asked for
  if (EPK_KERNELS[c->model][c->N](dgk::MODE_STAGE) && !(o && (o->elems_per_thread > 0 || o->groups_per_cta > 0))) {
    c->epk = true;
    c->k_rhs = EPK_KERNELS[c->model][c->N](dgk::MODE_RHS);
    c->k_stage = EPK_KERNELS[c->model][c->N](dgk::MODE_STAGE);
    c->k_ab3 = EPK_KERNELS[c->model][c->N](dgk::MODE_AB3);
    c->NT = 128;
    c->smem = 0;
    c->grid = (int)((c->K_active + 127) / 128);
    char buf[128];
    snprintf(buf, sizeof buf, "simt_elem_per_thread<%s,N=%d,threads=128,operators in constant memory>", c->model == DG_ACOUSTIC ? "acoustic" : "elastic", c->N);
    c->variant = buf;
    return;
  }
  // register blocking E and node groups G per CTA: at N <= 2 small batches win (more CTAs per SM hide the gather latency;
  // measured on the config-4 meshes: N = 1 E1 G16 1.34 ms vs E4 G32 2.70 ms per stage)
  const int E_auto = c->N == 1 ? 1 : (c->N == 2 ? (c->model == DG_ACOUSTIC ? 2 : 1) : (c->model == DG_ACOUSTIC ? 4 : 2));
  const int G_auto = c->N == 1 ? 16 : (c->N == 2 ? 8 : std::max(1, std::min(32, (224 + Np / 2) / Np)));
  int E = (o && o->elems_per_thread > 0) ? o->elems_per_thread : E_auto;
  int G = (o && o->groups_per_cta > 0) ? o->groups_per_cta : G_auto;
  if (!(o && o->groups_per_cta > 0)) {
    // keep the batch under ~64 KB of shared memory so several CTAs fit on an SM
    while (G > 1 && SMEM[c->model][c->N](G * E) > 64 * 1024) --G;
  }
  c->k_rhs = KERNELS[c->model][c->N](E, dgk::MODE_RHS);
  c->k_stage = KERNELS[c->model][c->N](E, dgk::MODE_STAGE);
  c->k_ab3 = KERNELS[c->model][c->N](E, dgk::MODE_AB3);
  if (!c->k_rhs || !c->k_stage || !c->k_ab3) throw std::invalid_argument("elems_per_thread not instantiated for this model");
  c->E = E;
  c->G = G;
  c->NT = ((G * Np + 31) / 32) * 32;
  if (c->NT > 1024) throw std::invalid_argument("groups_per_cta too large: more than 1024 threads");
  c->smem = SMEM[c->model][c->N](G * E);
  if (c->smem > 227 * 1024) throw std::invalid_argument("batch does not fit in shared memory");
  c->grid = (int)((c->K_active + (int64_t)G * E - 1) / ((int64_t)G * E));
  char buf[128];
  snprintf(buf, sizeof buf, "simt_fused<%s,N=%d,E=%d,G=%d,threads=%d,smem=%zu>", c->model == DG_ACOUSTIC ? "acoustic" : "elastic",
           c->N, E, G, c->NT, c->smem);
  c->variant = buf;
}

// 2-D TMA descriptors of a [K Nf][PT] fp32 device array for the tensor-core kernel's epilogue: boxes of `epi_cw`
// nodes x 32 rows ([0]) and x (Nf EB - 96) rows ([1]), 128 B / 64 B swizzle (tc3_kernels.cuh, epilogue)
typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                    const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
constexpr size_t TMAP_CACHE = 64;
// returns the descriptors BY VALUE: a later lookup may evict the entry (references into the map dangled)
std::array<CUtensorMap, 5> tensor_maps(dg_ctx *c, const void *ptr, bool pin = false) {
  auto it = c->tmaps.find(ptr);
  if (it != c->tmaps.end()) {
    it->second.stamp = ++c->tmap_clock;
    return it->second.m;
  }
  static encode_tiled_fn encode = nullptr;
  if (!encode) {
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn)
      throw std::runtime_error("cuda: cuTensorMapEncodeTiled is not available");
    encode = (encode_tiled_fn)fn;
  }
  if (c->tmaps.size() >= TMAP_CACHE) {           // evict the least recently used caller buffer (never a pinned one)
    auto victim = c->tmaps.end();
    for (auto jt = c->tmaps.begin(); jt != c->tmaps.end(); ++jt)
      if (!jt->second.pinned && (victim == c->tmaps.end() || jt->second.stamp < victim->second.stamp)) victim = jt;
    if (victim != c->tmaps.end()) c->tmaps.erase(victim);
  }
  std::array<CUtensorMap, 5> m;
  const int EB = TC3_INFO[c->model][c->N](1);
  const int rlast = c->NF * EB - 96;
  // [0], [1]: epilogue boxes of epi_cw nodes x 32 | rlast rows; [2]: field chunks of 16 nodes x 128 rows for the producers
  // (no-tile configurations); [3], [4]: the AB3 epilogue's boxes of epi_cw / 2 nodes.  Swizzle = the box's row length
  for (int h = 0; h < 5; ++h) {
    const int width = h == 2 ? 16 : (h < 2 ? c->epi_cw : c->epi_cw / 2);
    const cuuint64_t dims[2] = {(cuuint64_t)c->PT, (cuuint64_t)c->K_active * c->NF};   // (ghost rows are never loaded or stored by boxes)
    const cuuint64_t strides[1] = {(cuuint64_t)c->PT * 4};
    const int height = h == 2 ? 128 : ((h == 0 || h == 3) ? 32 : rlast);
    const cuuint32_t box[2] = {(cuuint32_t)width, (cuuint32_t)height};
    const cuuint32_t es[2] = {1, 1};
    const CUtensorMapSwizzle swz = width == 32 ? CU_TENSOR_MAP_SWIZZLE_128B : (width == 16 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_32B);
    const CUresult r = encode(&m[h], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void *>(ptr), dims, strides, box, es,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, swz,
                              CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) throw std::runtime_error("cuda: cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")");
  }
  c->tmaps.emplace(ptr, dg_ctx::TmapEntry{m, pin, ++c->tmap_clock});
  return m;
}

// elements per unit of work of the chosen kernel: element ranges of dg_stage_range start on multiples of it
int range_alignment(const dg_ctx *c) {
  if (c->tc3) return TC3_INFO[c->model][c->N](1);
  if (c->epk || c->rpt) return 1;
  return c->G * c->E;
}

// AB3 launches (kernel == c->k_ab3): hist1 = r^{m-1}, hist2 = r^{m-2} (inputs), rhs = the buffer that receives r^m
int launch_stage(dg_ctx *c, const void *kernel, const float *q_in, float *q_out, float *rhs, float a, float b, float dt,
                 cudaStream_t st, int64_t kbeg = 0, int64_t kend = -1, float *hist1 = nullptr, const float *hist2 = nullptr) {
  if (kend < 0) kend = c->K_active;
  if (kbeg >= kend) return DG_OK;
  dgk::StageParams p;
  p.q_in = q_in; p.q_out = q_out; p.res = hist1 ? hist1 : c->d_res; p.rhs = rhs; p.hist2 = hist2;
  p.DT = c->d_DT; p.LT = c->d_LT; p.geo = c->d_geo; p.nbr = c->d_nbr; p.fcode = c->d_fcode;
  p.fmask = c->d_fmask; p.nbrnode = c->d_nbrnode;
  p.K = (int)kend; p.kbeg = (int)kbeg; p.G = c->G; p.a = a; p.b = b; p.dt = dt;
  p.pflux = nullptr;
  if (c->surface) {                              // rows a4 + a5 by interfaces, into the face buffer the stage kernel lifts from
    dgk::IfaceParams ip;
    ip.q = q_in; ip.pflux = c->d_pflux; ip.geo = c->d_geo; ip.nbr = c->d_nbr; ip.fcode = c->d_fcode; ip.faces = c->d_ifaces;
    ip.fmask = c->d_fmask; ip.nbrnode = c->d_nbrnode; ip.nbrface = c->d_nbrface;
    ip.nint = c->n_int; ip.nbnd = c->n_bnd; ip.pitch = c->tc3 ? c->PT : c->Np;
    const long long nthreads = (long long)(c->n_int + c->n_bnd) * c->Nfp;
    void *iargs[] = {&ip};
    cudaError_t e = cudaLaunchKernel(c->k_iface, dim3((unsigned)((nthreads + 255) / 256)), dim3(256), iargs, 0, st);
    if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string("cuda: ") + cudaGetErrorString(e) + " launching the interface kernel");
    p.pflux = c->d_pflux;
    ++c->iface_launches;
  }
  int grid = c->grid;
  if (kbeg != 0 || kend != c->K_active) {
    const int unit = c->epk ? 128 : (c->rpt ? c->rpt_epc : range_alignment(c));
    grid = (int)((kend - kbeg + unit - 1) / unit);
  }
  if (c->rpt) {                                  // persistent warps: no more CTAs than the device holds at once
    if (c->rpt_cap == 0) {
      int per_sm = 0, sms = 0;
      cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, c->k_stage, c->NT, 0);
      if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device);
      if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string("cuda: ") + cudaGetErrorString(e) + " sizing the row-per-thread grid");
      c->rpt_cap = std::max(1, per_sm) * std::max(1, sms);
    }
    grid = std::min(grid, c->max_ctas > 0 ? std::min(c->rpt_cap, c->max_ctas) : c->rpt_cap);
  }
  dgk::Tc3Params tp3;
  void *args[] = {&p};
  if ((c->epk || c->rpt) && (((uintptr_t)q_in | (uintptr_t)q_out | (uintptr_t)rhs) & 15))
    return fail(DG_ERR_ARG, "device buffers must be 16-byte aligned");
  if (c->tc3) {
    if (((uintptr_t)q_in | (uintptr_t)q_out | (uintptr_t)rhs) & 15) return fail(DG_ERR_ARG, "device buffers must be 16-byte aligned");
    tp3.s = p;
    tp3.s.K = (int)c->K_active;                   // (the kernel bounds a ragged last batch by the advanced elements, ranges by batches)
    tp3.Bimg = c->d_Bimg;
    tp3.conn = c->d_conn;
    const int EB = range_alignment(c), nsplit = TC3_INFO[c->model][c->N](4);
    tp3.bbeg = (int)(kbeg / EB);
    tp3.nbatch = (int)((kend + EB - 1) / EB);
    int workers = std::max(1, std::min(tp3.nbatch - tp3.bbeg, c->num_sms / nsplit));
    if (c->max_ctas > 0) workers = std::max(1, std::min(workers, c->max_ctas / nsplit));
    grid = nsplit * workers;
    {
      try {
        const auto mi = tensor_maps(c, q_in), mr = tensor_maps(c, p.res), mo = tensor_maps(c, q_out ? q_out : rhs);
        for (int h = 0; h < 2; ++h) { tp3.tm_in[h] = mi[h]; tp3.tm_res[h] = mr[h]; tp3.tm_out[h] = mo[h]; }
        tp3.tm_u = mi[2];
        if (hist2) {
          const auto m2 = tensor_maps(c, hist2), m0 = tensor_maps(c, rhs);
          for (int h = 0; h < 2; ++h) {
            tp3.tm3_in[h] = mi[3 + h]; tp3.tm3_h1[h] = mr[3 + h]; tp3.tm3_h2[h] = m2[3 + h];
            tp3.tm3_r0[h] = m0[3 + h]; tp3.tm3_out[h] = mo[3 + h];
          }
        }
      } catch (const std::exception &e) {
        return fail(DG_ERR_CUDA, e.what());
      }
    }
    args[0] = &tp3;
  }
  cudaError_t e = cudaLaunchKernel(kernel, dim3(grid), dim3(c->NT), args, c->smem, st);
  if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string("cuda: ") + cudaGetErrorString(e) + " launching " + c->variant);
  return DG_OK;
}

int check_device_ctx(const dg_ctx *c) {
  if (!c) return fail(DG_ERR_ARG, "NULL context");
  if (c->device < 0) return fail(DG_ERR_CUDA, "host-only context: no device entry point is available (no CPU fallback)");
  return DG_OK;
}

#define DG_ENTER_DEVICE(c)                                \
  if (int e_ = check_device_ctx(c)) return e_;            \
  DeviceGuard guard_((c)->device);                        \
  if (!guard_.ok) return fail(DG_ERR_CUDA, "cuda: cannot select the context's device");   \
  (c)->iface_launches = 0

}  // namespace

// ================================================================================================
extern "C" {

const char *dg_last_error(void) { return g_err.c_str(); }

int dg_create(dg_ctx **out, const dg_mesh *mesh, int N, int model, const dg_materials *mat, const dg_options *opts) {
  if (!out) return fail(DG_ERR_ARG, "out is NULL");
  *out = nullptr;
  if (!mesh || !mat || !mesh->vxyz || !mesh->etov || !mat->rho || !mat->c_or_vp) return fail(DG_ERR_ARG, "NULL input pointer");
  if (N < 1 || N > 10) return fail(DG_ERR_ARG, "degree N must be in 1..10");
  if (model != DG_ACOUSTIC && model != DG_ELASTIC) return fail(DG_ERR_ARG, "unknown model");
  if (model == DG_ELASTIC && !mat->vs) return fail(DG_ERR_ARG, "elastic model needs vs");
  if (mesh->K <= 0 || mesh->nverts <= 0) return fail(DG_ERR_MESH, "mesh: empty mesh");
  if (mesh->K > 0x7FFFFFFF / 4) return fail(DG_ERR_MESH, "mesh: too many elements");
  dg_ctx *c = new (std::nothrow) dg_ctx();
  if (!c) return fail(DG_ERR_NOMEM, "out of host memory");
  try {
    c->N = N;
    c->model = model;
    c->NF = model == DG_ACOUSTIC ? 4 : 9;
    c->K = mesh->K;
    c->device = opts ? opts->device : 0;
    c->max_ctas = opts ? opts->max_ctas : 0;
    c->K_active = (opts && opts->owned_elements > 0) ? opts->owned_elements : c->K;
    if (c->K_active > c->K) throw std::invalid_argument("owned_elements exceeds the number of elements");
    c->surface = opts ? opts->surface : 0;
    if (c->surface != 0 && c->surface != 1) throw std::invalid_argument("surface must be 0 (element-centric) or 1 (interface-centric)");
    if (c->max_ctas < 0) throw std::invalid_argument("max_ctas must be >= 0");
    for (int64_t k = 0; k < c->K; ++k) {
      const double rho = mat->rho[k], cp = mat->c_or_vp[k];
      if (!(rho > 0.0) || !(cp > 0.0) || !std::isfinite(rho) || !std::isfinite(cp)) {
        delete c;
        return fail(DG_ERR_MATERIAL, "material: rho and c must be positive and finite");
      }
      if (model == DG_ELASTIC) {
        const double cs = mat->vs[k];
        if (!(cs > 0.0) || !(cp > cs * std::sqrt(4.0 / 3.0))) {
          delete c;
          return fail(DG_ERR_MATERIAL, "material: need vs > 0 and vp > vs*sqrt(4/3)");
        }
      }
    }
    dgh::build_refelem(N, c->ref);
    c->Np = c->ref.Np;
    c->Nfp = c->ref.Nfp;
    dgh::build_mesh(mesh->nverts, mesh->K, mesh->vxyz, mesh->etov, mesh->bc, c->mesh);
    if ((double)c->K * c->NF * c->Np >= 2147483647.0 * 4) throw std::runtime_error("mesh: field array too large");
    c->cmax.assign(mat->c_or_vp, mat->c_or_vp + c->K);
    choose_variant(c, opts);
    if (c->device >= 0) {
      DeviceGuard guard(c->device);              // dg_create leaves the caller's current device unchanged
      if (!guard.ok) throw std::runtime_error("cuda: cannot select device " + std::to_string(c->device));
      static_scratch_setup(c->device);           // (address of the static work memory of dg_step_static; allocates nothing)
      const int Np = c->Np, Nfp = c->Nfp;
      std::vector<float> DT((size_t)3 * Np * Np), LT((size_t)4 * Nfp * Np);
      const std::vector<double> *Dm[3] = {&c->ref.Dr, &c->ref.Ds, &c->ref.Dt};
      for (int d = 0; d < 3; ++d)
        for (int n = 0; n < Np; ++n)
          for (int m = 0; m < Np; ++m) DT[((size_t)d * Np + m) * Np + n] = (float)(*Dm[d])[(size_t)n * Np + m];
      for (int n = 0; n < Np; ++n)
        for (int j = 0; j < 4 * Nfp; ++j) LT[(size_t)j * Np + n] = (float)c->ref.LIFT[(size_t)n * 4 * Nfp + j];
      std::vector<float> geo;
      build_geo_records(c, mat, geo);
      std::vector<int> nbr((size_t)4 * c->K);
      for (size_t i = 0; i < nbr.size(); ++i) nbr[i] = c->mesh.nbr[i] >= 0 ? c->mesh.nbr[i] : -(int)c->mesh.bctag[i];
      std::vector<unsigned short> fmask(c->ref.fmask.begin(), c->ref.fmask.end());
      // device table indexed [f][g*6+s][i]
      std::vector<unsigned short> nbrnode(c->ref.nbrnode.begin(), c->ref.nbrnode.end());
      c->d_DT = upload(DT);
      c->d_LT = upload(LT);
      c->d_geo = upload(geo);
      c->d_nbr = upload(nbr);
      c->d_fcode = upload(c->mesh.fcode);
      c->d_fmask = upload(fmask);
      c->d_nbrnode = upload(nbrnode);
      if (c->epk) {
        std::vector<float> Dm((size_t)3 * Np * Np), Lm((size_t)Np * 4 * Nfp);
        const std::vector<double> *Ds3[3] = {&c->ref.Dr, &c->ref.Ds, &c->ref.Dt};
        for (int d = 0; d < 3; ++d)
          for (size_t i = 0; i < (size_t)Np * Np; ++i) Dm[(size_t)d * Np * Np + i] = (float)(*Ds3[d])[i];
        for (size_t i = 0; i < Lm.size(); ++i) Lm[i] = (float)c->ref.LIFT[i];
        std::vector<int> fm(c->ref.fmask.begin(), c->ref.fmask.end());
        const int rc = EPK_UPLOAD[c->model][c->N](Dm.data(), Lm.data(), nbrnode.data(), fm.data());
        if (rc == -1) throw std::runtime_error("element-per-thread kernel: face masks differ from the compile-time table");
        if (rc != 0) throw std::runtime_error(std::string("cuda: ") + cudaGetErrorString((cudaError_t)rc) + " uploading the operators to constant memory");
      }
      if (c->rpt) {
        std::vector<float> Dt((size_t)3 * Np * Np), Lt((size_t)4 * Nfp * Np);
        const std::vector<double> *Ds3[3] = {&c->ref.Dr, &c->ref.Ds, &c->ref.Dt};
        for (int m = 0; m < Np; ++m)
          for (int d = 0; d < 3; ++d)
            for (int n = 0; n < Np; ++n) Dt[((size_t)3 * m + d) * Np + n] = (float)(*Ds3[d])[(size_t)n * Np + m];
        for (int j = 0; j < 4 * Nfp; ++j)
          for (int n = 0; n < Np; ++n) Lt[(size_t)j * Np + n] = (float)c->ref.LIFT[(size_t)n * 4 * Nfp + j];
        const int rc = RPT_UPLOAD[c->model][c->N](Dt.data(), Lt.data());
        if (rc != 0) throw std::runtime_error(std::string("cuda: ") + cudaGetErrorString((cudaError_t)rc) + " uploading the operators to constant memory");
      }
      if (c->tc3) {
        const info_getter info = TC3_INFO[c->model][c->N];
        const int nsplit = info(4);
        std::vector<uint16_t> img;
        build_tc3_image(c->ref, info(2), nsplit, info(3), img);
        c->d_Bimg = upload(img);
        std::vector<int> conn((size_t)4 * c->K);
        for (size_t i = 0; i < conn.size(); ++i)
          conn[i] = c->mesh.nbr[i] >= 0 ? (int)(((uint32_t)c->mesh.nbr[i] << 5) | (c->mesh.fcode[i] & 31u)) : -(int)c->mesh.bctag[i];
        c->d_conn = upload(conn);
        CUDA_TRY(cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device));
        int workers = std::max(1, std::min(c->nbatch, c->num_sms / nsplit));        // persistent: one CTA per SM
        if (c->max_ctas > 0) workers = std::max(1, std::min(workers, c->max_ctas / nsplit));
        c->grid = nsplit * workers;
      }
      const size_t nq = (size_t)c->K * c->NF * Np;
      // the tensor-core kernel works on rows of pitch PT (16-byte aligned); when PT != Np the state lives in padded private
      // copies (pad columns are zero and stay zero) and is converted on entry / exit of every API call
      const size_t nqp = c->tc3 ? (size_t)c->K * c->NF * c->PT : nq;
      CUDA_TRY(cudaMalloc(&c->d_res, nqp * sizeof(float)));
      CUDA_TRY(cudaMalloc(&c->d_q2, nqp * sizeof(float)));
      CUDA_TRY(cudaMemset(c->d_q2, 0, nqp * sizeof(float)));
      if (c->tc3 && c->PT != Np) {
        CUDA_TRY(cudaMalloc(&c->d_qa, nqp * sizeof(float)));
        CUDA_TRY(cudaMemset(c->d_qa, 0, nqp * sizeof(float)));
      }
      for (float *&h : c->d_hist) {             // AB3 history, in the kernel's own row pitch
        CUDA_TRY(cudaMalloc(&h, nqp * sizeof(float)));
        CUDA_TRY(cudaMemset(h, 0, nqp * sizeof(float)));
      }
      CUDA_TRY(cudaMemset(c->d_res, 0, nqp * sizeof(float)));
      if (c->surface) {
        // one entry per interface (listed by the side with the smaller element number), boundary faces behind
        std::vector<int> faces, bnd;
        for (int64_t k = 0; k < c->K; ++k)
          for (int f = 0; f < 4; ++f) {
            const int32_t nb = c->mesh.nbr[4 * k + f];
            if (nb < 0) bnd.push_back((int)(4 * k + f));
            else if (nb > k) faces.push_back((int)(4 * k + f));
          }
        c->n_int = (int)faces.size();
        c->n_bnd = (int)bnd.size();
        faces.insert(faces.end(), bnd.begin(), bnd.end());
        c->d_ifaces = upload(faces);
        std::vector<unsigned short> nbrface(c->ref.nbrface.begin(), c->ref.nbrface.end());
        c->d_nbrface = upload(nbrface);
        CUDA_TRY(cudaMalloc(&c->d_pflux, (size_t)c->K * c->NF * 4 * Nfp * sizeof(float)));
        c->k_iface = IFACE_KERNELS[c->model][c->N]();
        c->variant += " + interface-centric surface kernel";
      }
      if (c->tc3) {                              // descriptors of the library's own buffers: encoded once, never evicted
        tensor_maps(c, c->d_res, true);
        tensor_maps(c, c->d_q2, true);
        if (c->d_qa) tensor_maps(c, c->d_qa, true);
        for (float *h : c->d_hist) tensor_maps(c, h, true);
      }
      CUDA_TRY(cudaFuncSetAttribute(c->k_rhs, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem));
      CUDA_TRY(cudaFuncSetAttribute(c->k_stage, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem));
      CUDA_TRY(cudaFuncSetAttribute(c->k_ab3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->smem));
      CUDA_TRY(cudaDeviceSynchronize());
    }
  } catch (const std::invalid_argument &e) {
    free_device(c);
    delete c;
    return fail(DG_ERR_ARG, e.what());
  } catch (const std::bad_alloc &) {
    free_device(c);
    delete c;
    return fail(DG_ERR_NOMEM, "out of host memory");
  } catch (const std::exception &e) {
    const std::string msg = e.what();
    free_device(c);
    delete c;
    if (msg.rfind("cuda:", 0) == 0) return fail(msg.find("out of memory") != std::string::npos ? DG_ERR_NOMEM : DG_ERR_CUDA, msg);
    if (msg.rfind("mesh:", 0) == 0) return fail(DG_ERR_MESH, msg);
    return fail(DG_ERR_ARG, msg);
  }
  *out = c;
  return DG_OK;
}

int dg_destroy(dg_ctx *c) {
  if (!c) return fail(DG_ERR_ARG, "NULL context");
  free_device(c);
  delete c;
  return DG_OK;
}

int dg_num_fields(const dg_ctx *c) { return c ? c->NF : fail(DG_ERR_ARG, "NULL context"); }
int dg_np(const dg_ctx *c) { return c ? c->Np : fail(DG_ERR_ARG, "NULL context"); }
int dg_nfp(const dg_ctx *c) { return c ? c->Nfp : fail(DG_ERR_ARG, "NULL context"); }
int64_t dg_num_elements(const dg_ctx *c) { return c ? c->K : (int64_t)fail(DG_ERR_ARG, "NULL context"); }
int dg_last_launch_count(const dg_ctx *c) { return c ? c->last_launches : fail(DG_ERR_ARG, "NULL context"); }
const char *dg_variant_name(const dg_ctx *c) { return c ? c->variant.c_str() : ""; }

int dg_node_coords(const dg_ctx *c, double *xyz) {
  if (!c || !xyz) return fail(DG_ERR_ARG, "NULL argument");
  const int Np = c->Np;
  for (int64_t k = 0; k < c->K; ++k) {
    const double *v = &c->mesh.verts[12 * k];
    for (int n = 0; n < Np; ++n) {
      const double r = c->ref.r[n], s = c->ref.s[n], t = c->ref.t[n];
      for (int d = 0; d < 3; ++d)
        xyz[((size_t)k * Np + n) * 3 + d] = 0.5 * (-(1.0 + r + s + t) * v[d] + (1.0 + r) * v[3 + d] + (1.0 + s) * v[6 + d] + (1.0 + t) * v[9 + d]);
    }
  }
  return DG_OK;
}

double dg_stable_dt(const dg_ctx *c, double cfl) {
  if (!c || !(cfl > 0.0)) return (double)fail(DG_ERR_ARG, "bad argument");
  double worst = 0.0;
  for (int64_t k = 0; k < c->K; ++k) {
    double fs = 0.0;
    for (int f = 0; f < 4; ++f) fs = std::max(fs, c->mesh.fscale[4 * k + f]);
    worst = std::max(worst, c->cmax[k] * fs);
  }
  return cfl / ((c->N + 1.0) * (c->N + 1.0) * worst);
}

int dg_reference_operators(const dg_ctx *c, double *Dr, double *Ds, double *Dt, double *LIFT, double *rst, int32_t *fmask) {
  if (!c) return fail(DG_ERR_ARG, "NULL context");
  const size_t nn = (size_t)c->Np * c->Np;
  if (Dr) std::memcpy(Dr, c->ref.Dr.data(), nn * sizeof(double));
  if (Ds) std::memcpy(Ds, c->ref.Ds.data(), nn * sizeof(double));
  if (Dt) std::memcpy(Dt, c->ref.Dt.data(), nn * sizeof(double));
  if (LIFT) std::memcpy(LIFT, c->ref.LIFT.data(), (size_t)c->Np * 4 * c->Nfp * sizeof(double));
  if (rst)
    for (int n = 0; n < c->Np; ++n) {
      rst[3 * n + 0] = c->ref.r[n];
      rst[3 * n + 1] = c->ref.s[n];
      rst[3 * n + 2] = c->ref.t[n];
    }
  if (fmask) std::memcpy(fmask, c->ref.fmask.data(), (size_t)4 * c->Nfp * sizeof(int32_t));
  return DG_OK;
}

int dg_geometry(const dg_ctx *c, double *G, double *J, double *nrm, double *fscale) {
  if (!c) return fail(DG_ERR_ARG, "NULL context");
  if (G) std::memcpy(G, c->mesh.G.data(), c->mesh.G.size() * sizeof(double));
  if (J) std::memcpy(J, c->mesh.J.data(), c->mesh.J.size() * sizeof(double));
  if (nrm) std::memcpy(nrm, c->mesh.nrm.data(), c->mesh.nrm.size() * sizeof(double));
  if (fscale) std::memcpy(fscale, c->mesh.fscale.data(), c->mesh.fscale.size() * sizeof(double));
  return DG_OK;
}

int dg_connectivity(const dg_ctx *c, int32_t *elemP, int32_t *nodeP, int8_t *bctag) {
  if (!c) return fail(DG_ERR_ARG, "NULL context");
  const int Nfp = c->Nfp;
  for (int64_t k = 0; k < c->K; ++k)
    for (int f = 0; f < 4; ++f) {
      const int32_t nb = c->mesh.nbr[4 * k + f];
      for (int i = 0; i < Nfp; ++i) {
        const size_t o = ((size_t)k * 4 + f) * Nfp + i;
        if (nb >= 0) {
          const int code = c->mesh.fcode[4 * k + f];
          if (elemP) elemP[o] = nb;
          if (nodeP) nodeP[o] = c->ref.nbrnode[((size_t)f * 24 + code) * Nfp + i];
        } else {
          if (elemP) elemP[o] = (int32_t)k;
          if (nodeP) nodeP[o] = c->ref.fmask[f * Nfp + i];
        }
      }
      if (bctag) bctag[4 * k + f] = c->mesh.bctag[4 * k + f];
    }
  return DG_OK;
}

// caller layout [K Nf][Np] <-> the tensor-core kernel's private layout [K Nf][PT] (pad columns stay zero)
static bool padded(const dg_ctx *c) { return c->tc3 && c->PT != c->Np; }
static int copy_rows(dg_ctx *c, float *dst, int dpitch, const float *src, int spitch, cudaStream_t st) {
  const size_t n = (size_t)c->K * c->NF * c->Np;
  const int blocks = (int)std::min<size_t>((n + 255) / 256, (size_t)148 * 32);
  dgk::repitch_kernel<<<blocks, 256, 0, st>>>(dst, dpitch, src, spitch, c->Np, n);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string("cuda: ") + cudaGetErrorString(e) + " in the layout conversion");
  return DG_OK;
}
// r(q) -> d_out (caller layout); adds the number of launches / copies enqueued to `launches`
static int eval_rhs(dg_ctx *c, const float *d_q, float *d_out, cudaStream_t st, int &launches) {
  if (!padded(c)) {
    launches += 1;
    return launch_stage(c, c->k_rhs, d_q, nullptr, d_out, 0.f, 0.f, 0.f, st);
  }
  if (int e = copy_rows(c, c->d_qa, c->PT, d_q, c->Np, st)) return e;
  if (int e = launch_stage(c, c->k_rhs, c->d_qa, nullptr, c->d_q2, 0.f, 0.f, 0.f, st)) return e;
  launches += 3;
  return copy_rows(c, d_out, c->Np, c->d_q2, c->PT, st);
}

int dg_rhs(dg_ctx *c, const float *d_q, float *d_rhs, void *stream) {
  DG_ENTER_DEVICE(c);
  if (!d_q || !d_rhs) return fail(DG_ERR_ARG, "NULL device pointer");
  if (d_q == d_rhs) return fail(DG_ERR_ARG, "dg_rhs: d_q and d_rhs must differ");
  c->last_launches = 0;
  const int rc = eval_rhs(c, d_q, d_rhs, (cudaStream_t)stream, c->last_launches);
  c->last_launches += c->iface_launches;
  return rc;
}

int dg_run(dg_ctx *c, float *d_q, float dt, int nsteps, void *stream) {
  DG_ENTER_DEVICE(c);
  if (!d_q || nsteps < 0) return fail(DG_ERR_ARG, "bad argument");
  cudaStream_t st = (cudaStream_t)stream;
  int launches = 0;
  if (padded(c)) {
    // private padded state: convert once on entry and once on exit, the 5 nsteps stage kernels ping-pong d_qa <-> d_q2
    if (nsteps > 0) {
      if (int e = copy_rows(c, c->d_qa, c->PT, d_q, c->Np, st)) return e;
      float *cur = c->d_qa, *oth = c->d_q2;
      for (int s = 0; s < nsteps; ++s)
        for (int i = 0; i < 5; ++i) {
          if (int e = launch_stage(c, c->k_stage, cur, oth, nullptr, (float)RK_A[i], (float)RK_B[i], dt, st)) return e;
          std::swap(cur, oth);
        }
      if (int e = copy_rows(c, d_q, c->Np, cur, c->PT, st)) return e;
      launches = 5 * nsteps + 2;
    }
    c->last_launches = launches + c->iface_launches;
    return DG_OK;
  }
  float *cur = d_q, *oth = c->d_q2;
  for (int s = 0; s < nsteps; ++s)
    for (int i = 0; i < 5; ++i) {
      if (int e = launch_stage(c, c->k_stage, cur, oth, nullptr, (float)RK_A[i], (float)RK_B[i], dt, st)) return e;
      std::swap(cur, oth);
      ++launches;
    }
  if (cur != d_q) {
    cudaError_t e = cudaMemcpyAsync(d_q, cur, (size_t)c->K * c->NF * c->Np * sizeof(float), cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string("cuda: ") + cudaGetErrorString(e));
    ++launches;
  }
  c->last_launches = launches + c->iface_launches;
  return DG_OK;
}

int dg_step(dg_ctx *c, float *d_q, float dt, void *stream) { return dg_run(c, d_q, dt, 1, stream); }

// One LSRK step like dg_step, with the residual and the ping-pong state (and, for the padded-row degrees of the tensor-core
// kernel, the private padded copy of q) in dg_static_scratch instead of the context's buffers.  No cudaMalloc / cudaFree
// and no allocating library call: memset, the stage kernels, the row re-pitch kernel and one device copy.
int dg_step_static(dg_ctx *c, float *d_q, float dt, void *stream) {
  DG_ENTER_DEVICE(c);
  if (!d_q) return fail(DG_ERR_ARG, "NULL device pointer");
  if (c->device >= STATIC_SCRATCH_MAX_DEVICES) return fail(DG_ERR_ARG, "dg_step_static: device ordinal beyond the address table");
  static_scratch_setup(c->device);                // (normally a no-op: resolved by dg_create)
  unsigned char *base = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_scratch_mu);
    if (g_scratch_state[c->device] != 1)
      return fail(DG_ERR_CUDA, std::string("cuda: ") + cudaGetErrorString((cudaError_t)(-g_scratch_state[c->device])) +
                                   " resolving the address of the static work memory (cudaGetSymbolAddress)");
    base = g_scratch_ptr[c->device];
  }
  const bool pad = padded(c);
  const size_t pitch = c->tc3 ? (size_t)c->PT : (size_t)c->Np;
  const size_t arr = ((size_t)c->K * c->NF * pitch * sizeof(float) + 255) / 256 * 256;     // one array, 256-byte granules
  const size_t narr = pad ? 3 : 2, need = narr * arr;
  if (need > (size_t)DG_STATIC_SCRATCH_BYTES)
    return fail(DG_ERR_ARG, "dg_step_static: this context needs " + std::to_string(need) + " bytes of work memory (" + std::to_string(narr) +
                                " arrays of K Nf Np floats), the static array holds DG_STATIC_SCRATCH_BYTES = " +
                                std::to_string((size_t)DG_STATIC_SCRATCH_BYTES) + ": use dg_step");
  cudaStream_t st = (cudaStream_t)stream;
  // the array keeps the last call's contents: everything this call uses starts from zero (the pad columns of padded rows
  // must be zero, and stay zero; the residual is overwritten by stage 1, A_1 = 0)
  cudaError_t e = cudaMemsetAsync(base, 0, need, st);
  if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string("cuda: ") + cudaGetErrorString(e) + " clearing the static work memory");
  float *res = reinterpret_cast<float *>(base), *q2 = reinterpret_cast<float *>(base + arr);
  float *qa = pad ? reinterpret_cast<float *>(base + 2 * arr) : d_q;
  int launches = 1;
  if (pad) {
    if (int rc = copy_rows(c, qa, c->PT, d_q, c->Np, st)) return rc;
    ++launches;
  }
  float *cur = qa, *oth = q2;
  for (int i = 0; i < 5; ++i) {
    if (int rc = launch_stage(c, c->k_stage, cur, oth, nullptr, (float)RK_A[i], (float)RK_B[i], dt, st, 0, -1, res)) return rc;
    std::swap(cur, oth);
    ++launches;
  }
  if (pad) {
    if (int rc = copy_rows(c, d_q, c->Np, cur, c->PT, st)) return rc;
  } else {
    e = cudaMemcpyAsync(d_q, cur, (size_t)c->K * c->NF * c->Np * sizeof(float), cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string("cuda: ") + cudaGetErrorString(e));
  }
  c->last_launches = launches + 1 + c->iface_launches;
  return DG_OK;
}

int dg_stage(dg_ctx *c, const float *d_q_in, float *d_q_out, float a, float b, float dt, void *stream) {
  DG_ENTER_DEVICE(c);
  if (!d_q_in || !d_q_out) return fail(DG_ERR_ARG, "NULL device pointer");
  if (d_q_in == d_q_out) return fail(DG_ERR_ARG, "dg_stage: d_q_in and d_q_out must differ (neighbours read the stage input)");
  cudaStream_t st = (cudaStream_t)stream;
  if (!padded(c)) {
    c->last_launches = 1 + c->surface;
    return launch_stage(c, c->k_stage, d_q_in, d_q_out, nullptr, a, b, dt, st);
  }
  if (int e = copy_rows(c, c->d_qa, c->PT, d_q_in, c->Np, st)) return e;
  if (int e = launch_stage(c, c->k_stage, c->d_qa, c->d_q2, nullptr, a, b, dt, st)) return e;
  c->last_launches = 3 + c->surface;
  return copy_rows(c, d_q_out, c->Np, c->d_q2, c->PT, st);
}

static int halo_move(dg_ctx *c, float *d_q, const int32_t *d_faces, int64_t nfaces, float *d_buf, void *stream, bool pack) {
  if (!d_q || !d_buf || !d_faces || nfaces < 0) return fail(DG_ERR_ARG, "bad argument");
  c->last_launches = 0;
  if (nfaces == 0) return DG_OK;
  const size_t n = (size_t)nfaces * c->NF * c->Nfp;
  const int blocks = (int)std::min<size_t>((n + 255) / 256, (size_t)148 * 16);
  if (pack) dgk::halo_kernel<true><<<blocks, 256, 0, (cudaStream_t)stream>>>(d_q, d_buf, d_faces, c->d_fmask, c->NF, c->Np, c->Nfp, n);
  else dgk::halo_kernel<false><<<blocks, 256, 0, (cudaStream_t)stream>>>(d_q, d_buf, d_faces, c->d_fmask, c->NF, c->Np, c->Nfp, n);
  if (cudaGetLastError() != cudaSuccess) return fail(DG_ERR_CUDA, "cuda: halo kernel launch failed");
  c->last_launches = 1;
  return DG_OK;
}

int dg_halo_pack(dg_ctx *c, const float *d_q, const int32_t *d_faces, int64_t nfaces, float *d_buf, void *stream) {
  DG_ENTER_DEVICE(c);
  return halo_move(c, const_cast<float *>(d_q), d_faces, nfaces, d_buf, stream, true);
}

int dg_halo_unpack(dg_ctx *c, float *d_q, const int32_t *d_faces, int64_t nfaces, const float *d_buf, void *stream) {
  DG_ENTER_DEVICE(c);
  return halo_move(c, d_q, d_faces, nfaces, const_cast<float *>(d_buf), stream, false);
}

int64_t dg_num_owned_elements(const dg_ctx *c) { return c ? c->K_active : (int64_t)fail(DG_ERR_ARG, "NULL context"); }

int dg_range_alignment(const dg_ctx *c) { return c ? range_alignment(c) : fail(DG_ERR_ARG, "NULL context"); }

int dg_stage_range(dg_ctx *c, const float *d_q_in, float *d_q_out, float a, float b, float dt, int64_t k_begin, int64_t k_end,
                   void *stream) {
  DG_ENTER_DEVICE(c);
  if (!d_q_in || !d_q_out) return fail(DG_ERR_ARG, "NULL device pointer");
  if (d_q_in == d_q_out) return fail(DG_ERR_ARG, "dg_stage_range: d_q_in and d_q_out must differ");
  if (k_begin < 0 || k_end > c->K_active || k_begin > k_end) return fail(DG_ERR_ARG, "dg_stage_range: need 0 <= k_begin <= k_end <= K (owned elements)");
  if (k_begin % range_alignment(c) != 0 || (k_end % range_alignment(c) != 0 && k_end != c->K_active))
    return fail(DG_ERR_ARG, "dg_stage_range: k_begin and k_end must be multiples of dg_range_alignment() (k_end may be K)");
  if (padded(c)) return fail(DG_ERR_ARG, "dg_stage_range: not available for degrees whose rows the library pads (N = 2, 4, 8, 10 on the tensor-core variant); create the context with variant = 1");
  c->last_launches = k_begin < k_end ? 1 + c->surface : 0;
  return launch_stage(c, c->k_stage, d_q_in, d_q_out, nullptr, a, b, dt, (cudaStream_t)stream, k_begin, k_end);
}

int dg_element_dt(const dg_ctx *c, double cfl, double *dt_host) {
  if (!c || !dt_host || !(cfl > 0.0)) return fail(DG_ERR_ARG, "bad argument");
  for (int64_t k = 0; k < c->K; ++k) {
    double fs = 0.0;
    for (int f = 0; f < 4; ++f) fs = std::max(fs, c->mesh.fscale[4 * k + f]);
    dt_host[k] = cfl / ((c->N + 1.0) * (c->N + 1.0) * c->cmax[k] * fs);
  }
  return DG_OK;
}

int dg_ab3_reset(dg_ctx *c, void *stream) {
  DG_ENTER_DEVICE(c);
  (void)stream;
  c->nhist = 0;                                  // the next two steps are start-up steps again
  c->hist_head = 0;
  return DG_OK;
}

// nsteps steps of PAPER.md eq. (4).  Steady state: ONE fused kernel per step (r(q), the AB3 combination and the rotation of
// the history R_0, R_-1, R_-2 of Table 1, by pointer), q ping-pong as in dg_run.  Start-up (DESIGN.md reading
// Q21): while fewer than two earlier right-hand sides are on record a step is r(q) into the history + one LSRK(5,4) step.
int dg_ab3_run(dg_ctx *c, float *d_q, float dt, int nsteps, void *stream) {
  DG_ENTER_DEVICE(c);
  if (!d_q || nsteps < 0) return fail(DG_ERR_ARG, "bad argument");
  cudaStream_t st = (cudaStream_t)stream;
  int launches = 0;
  c->last_launches = 0;
  if (nsteps == 0) return DG_OK;
  float *cur = d_q, *oth = c->d_q2;
  if (padded(c)) {
    if (int e = copy_rows(c, c->d_qa, c->PT, d_q, c->Np, st)) return e;
    cur = c->d_qa;
    ++launches;
  }
  const float c0 = dt * (23.f / 12.f), c1 = dt * (-16.f / 12.f), c2 = dt * (5.f / 12.f);
  for (int s = 0; s < nsteps; ++s) {
    float *h1 = c->d_hist[c->hist_head], *h2 = c->d_hist[(c->hist_head + 1) % 3], *r0 = c->d_hist[(c->hist_head + 2) % 3];
    if (c->nhist < 2) {
      if (int e = launch_stage(c, c->k_rhs, cur, nullptr, r0, 0.f, 0.f, 0.f, st)) return e;
      for (int i = 0; i < 5; ++i) {
        if (int e = launch_stage(c, c->k_stage, cur, oth, nullptr, (float)RK_A[i], (float)RK_B[i], dt, st)) return e;
        std::swap(cur, oth);
      }
      launches += 6;
      ++c->nhist;
    } else {
      if (int e = launch_stage(c, c->k_ab3, cur, oth, r0, c1, c2, c0, st, 0, -1, h1, h2)) return e;
      std::swap(cur, oth);
      ++launches;
    }
    c->hist_head = (c->hist_head + 2) % 3;       // r^m becomes r^{m-1}, r^{m-1} becomes r^{m-2}
  }
  if (padded(c)) {
    if (int e = copy_rows(c, d_q, c->Np, cur, c->PT, st)) return e;
    ++launches;
  } else if (cur != d_q) {
    cudaError_t e = cudaMemcpyAsync(d_q, cur, (size_t)c->K * c->NF * c->Np * sizeof(float), cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return fail(DG_ERR_CUDA, std::string("cuda: ") + cudaGetErrorString(e));
    ++launches;
  }
  c->last_launches = launches + c->iface_launches;
  return DG_OK;
}

int dg_ab3_step(dg_ctx *c, float *d_q, float dt, void *stream) { return dg_ab3_run(c, d_q, dt, 1, stream); }

#ifdef DG_PROF
// development builds only (-DDG_PROF; declared in dg_prof.h, not in include/dg.h)
int dg_prof_read(dg_ctx *c, long long *out) {
  typedef int (*rd)(long long *);
  static const rd R[2][11] = {DG_ROW(0, dgk_prof_read_), DG_ROW(1, dgk_prof_read_)};
  cudaDeviceSynchronize();
  return R[c->model][c->N](out);
}
#endif

}  // extern "C"
