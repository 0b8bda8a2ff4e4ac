// Pipelined warp-specialised tensor-core stage kernel of libdg (sm_100a), variant 4: "tc_pipe".
//
// One contraction per batch of 32 acoustic / 14 elastic elements (up to 128 (element,
// field) rows = TMEM lanes)
//
//     R[row][n] = sum_k  A[row][k] * B[n][k]
//
// k = (D_j, node m): A = pre-combined (rows a1 + a3), vertex-mean shifted fields, B = D_j[n][m]  (row a2;
// PAPER.md:171, eq. (9)-(10) P:191-204);  k = face node: A = penalty terms times g^sur (rows a4, a5), B = LIFT
// (row a6); LSRK update (row a7) in the epilogue -- in BF16x3 split precision (six kind::f16 MMAs
// per 16-wide k-step, two fp32 accumulators in TMEM), but with every stage of the path decoupled so that the
// gather latency, the field-tile load and the epilogue overlap the MMAs of neighbouring batches:
//
//   * a loader warp streams the batch's field tile, geometric records and packed connectivity into a
//     double-buffered shared-memory slot with bulk async copies (one batch ahead) and prefetches the batch's
//     residual into L2 for the epilogue; where the tile does not fit in shared memory (N >= 8) it streams the
//     fields as 2-D TMA boxes of 16 nodes x 128 rows through a ring instead;
//   * the flux warps (face gather a4 + penalty a5) work through a ring of chunks of 16 (N <= 3) or 32 face nodes,
//     several chunks -- and, with two tile slots, one batch -- ahead of the producers; exterior traces of
//     neighbours inside the batch come from the shared-memory tile, the others from L2; all gathers of a chunk
//     are issued before the first use;
//   * the epilogue moves chunks of 32 rows x 16|32 nodes as swizzled 2-D TMA boxes (res / q in two chunks ahead,
//     results out through the same staging buffers) and updates in the TMEM-native layout (thread = row);
//   * every array the kernel touches has 16-byte aligned rows (pitch PT = Np rounded up to 4; dg_api.cu keeps
//     padded private copies of the state where Np % 4 != 0);
//   * degrees whose panel exceeds the TMEM budget (N >= 9) split the output nodes over NSPLIT = 2 CTAs
//     (each CTA owns half of the operator rows and its own accumulators).
//
// Warp roles (736 threads): 0-3 epilogue, 4-11 producers (lane = row; tcgen05.st into the TMEM A ring),
// 12-19 flux, 20 operator stream (cp.async.bulk ring), 21 MMA issue + TMEM allocation, 22 tile loader.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "flux.cuh"
#include "kernels.cuh"
#include "tc_common.cuh"

namespace dgk {

constexpr int T3_FLUXW = 8;           // flux warps
constexpr int T3_W_OPS = 12 + T3_FLUXW, T3_W_MMA = T3_W_OPS + 1, T3_W_LOAD = T3_W_OPS + 2;   // single-warp roles
constexpr int T3_THREADS = (T3_W_LOAD + 1) * 32;
constexpr int T3_NU = 4;             // field chunk ring stages (shared memory; only when the whole tile does not fit)
constexpr int T3_UCH = 128 * 16 * 4;  // bytes of one field chunk: 128 rows x 16 nodes
constexpr int T3_ASTRIDE = 24;       // TMEM columns per A stage: 3 pieces x 8 columns (16 bf16)
constexpr int T3_SMEM_LIMIT = 227 * 1024 - 512;

template <int MODEL, int N>
struct T3 {
  using D = Deg<N>;
  static constexpr int NP = D::NP, NFP = D::NFP, NFACE = D::NFACE;
  static constexpr int NF = MODEL == 0 ? 4 : 9;
  static constexpr int NGEO = MODEL == 0 ? GEO_AC : GEO_EL;
  static constexpr int EB = MODEL == 0 ? 32 : 14;              // elements per batch
  static constexpr int NR = EB * NF;                           // valid rows (<= 128)
  static constexpr int PT = (NP + 3) / 4 * 4;                  // row pitch of q / res / rhs (floats): rows 16-byte aligned
  static constexpr int NC = (NP + 15) / 16 * 16;               // output nodes, padded
  static constexpr int NSPLIT = NC > 176 ? 2 : 1;              // CTAs sharing one batch (output-node halves)
  static constexpr int NCH = NC / NSPLIT;                      // MMA N of one CTA
  static constexpr int NB = NCH >= 144 ? 3 : 4;                // operator ring stages (shared memory)
  // flux chunks: 32 face nodes (two k-steps; four tasks in flight per flux thread) from N = 4 up, 16 below, where a
  // batch has only two or three k-steps of face nodes (same-box A/B: N = 3 is 7 % slower with 32, acoustic N = 4 6 %
  // faster, N = 10 9 % faster)
  static constexpr int FCH = N >= 4 ? 32 : 16;
  static constexpr int FLS = FCH + 4;                          // floats per row of a chunk (80 / 144-byte rows: conflict-free float4)
  static constexpr int NFL = FCH == 16 ? 4 : (NC >= 176 ? 4 : 3);                // flux chunk ring stages: enough to cover the producers' volume phase
  static constexpr int NG = (NP + 15) / 16;                    // node chunks of 16
  static constexpr int NH = (NFACE + 15) / 16;                 // face-node k-steps of 16
  static constexpr int NHC = (NFACE + FCH - 1) / FCH;          // flux chunks
  static constexpr int NSTEP = 3 * NG + NH;                    // k-steps of 16 per batch
  static constexpr int NSETS = (4 * NCH + 3 * T3_ASTRIDE <= 512) ? 2 : 1;   // accumulator sets
  static constexpr int ABASE = NSETS * 2 * NCH;                // first TMEM column of the A ring
  static constexpr int NA_ = (512 - ABASE) / T3_ASTRIDE;
  static constexpr int NA = NA_ > 9 ? 9 : NA_;                 // A ring stages
  static constexpr int BSTAGE = 96 * NCH;                      // bytes: [3 pieces][2 kc][NCH][8] bf16
  static constexpr int TILE_RAW = EB * NF * PT * 4;            // bytes of the batch's fields (multiple of 16)
  static constexpr int META = EB * NGEO * 4 + EB * 16;         // geometric records + packed connectivity
  static constexpr int FLUX_SLOT = 128 * FLS * 4;
  static constexpr int CW = NC >= 128 ? 16 : 32;               // epilogue chunk width (output nodes)
  static constexpr int NES = CW == 16 ? 3 : 2;                 // epilogue staging stages
  static constexpr int SCR = 4 * NES * 2 * 32 * CW * 4;        // per epilogue warp: [stage][res | q][32 rows][CW] floats (swizzled)
  static constexpr int NBAR = 2 * NA + 2 * NB + 2 * NFL + 4 + 4 + 12 + 2 * T3_NU;
  // neighbour-node table [4][24][NFP] and face mask [4 NFP] (uint16) for the flux warps: in shared memory, so that the
  // exterior-trace gather is one dependent load (connectivity -> address) instead of two through L2 (the L1 left beside
  // ~210 KB of shared memory does not hold the table: ncu showed 28 % of the flux warps' stall samples on these loads)
  static constexpr int TAB = ((96 + 4) * NFP * 2 + 15) / 16 * 16;
  static constexpr int FIXED = NB * BSTAGE + NFL * FLUX_SLOT + SCR + TAB + NBAR * 8 + 16 + 1024;
  static constexpr int TILE_SLOT = TILE_RAW;
  static constexpr bool TILE = FIXED + TILE_SLOT + META <= T3_SMEM_LIMIT;   // field tile staged in shared memory
  static constexpr int NQ = !TILE ? 2 : (FIXED + 2 * (TILE_SLOT + META) <= T3_SMEM_LIMIT ? 2 : 1);
  static constexpr int SLOT = (TILE ? TILE_SLOT : 0) + META;   // bytes of one tile slot
  static constexpr int URING = TILE ? 0 : T3_NU * T3_UCH;      // field chunk ring (TMA boxes of 16 nodes x 128 rows)
  // shared-memory carve-up (bytes)
  static constexpr int OFF_B = 0;
  static constexpr int OFF_FLUX = OFF_B + NB * BSTAGE;
  static constexpr int OFF_SCR = OFF_FLUX + NFL * FLUX_SLOT;
  static constexpr int OFF_U = OFF_SCR + SCR;
  static constexpr int OFF_SLOT = OFF_U + URING;
  static constexpr int OFF_TAB = OFF_SLOT + NQ * SLOT;
  static constexpr int OFF_BAR = OFF_TAB + TAB;
  static constexpr int SMEM = OFF_BAR + NBAR * 8 + 16 + 1024;  // + slack for the 1024-byte alignment (swizzled TMA boxes)
  // exterior traces of neighbours inside the batch are read from the shared-memory tile (elastic from N = 3, acoustic from
  // N = 6): below, the uniform all-L2 gather is faster than the divergent two-path one (same-box A/B: C2 0.573 -> 0.564 ms,
  // elastic N = 2 2.87 -> 2.81 ms; elastic N = 3..5 are 1-2 % slower without the shared-memory path)
  static constexpr bool INBATCH = TILE && (MODEL == 1 ? N >= 3 : N >= 6);
  static constexpr int TPT = (EB * FCH + T3_FLUXW * 32 - 1) / (T3_FLUXW * 32);           // flux tasks per thread and chunk
  static_assert(NR <= 128 && NCH <= 256 && NCH % 16 == 0, "one M tile, legal MMA N");
  static_assert(NA >= 3, "A ring too small");
  static_assert((T3_FLUXW * 32) % FCH == 0, "a flux thread keeps its face node across its tasks");
  static_assert(SMEM <= 227 * 1024, "shared memory");
  static_assert(SLOT % 16 == 0 && BSTAGE % 16 == 0, "bulk copy alignment");
  static_assert(OFF_SCR % (CW == 32 ? 1024 : 512) == 0 && (32 * CW * 4) % (CW == 32 ? 1024 : 512) == 0,
                "swizzled TMA staging buffers: 1024-byte (128 B swizzle) / 512-byte (64 B swizzle) alignment");
  static_assert(OFF_U % 512 == 0 && T3_UCH % 512 == 0, "field chunk ring: 64 B swizzle atoms are 512 bytes");
};

// Optional role timeline (build with -DDG_PROF): every warp accumulates the cycles it spends in each kind of
// mbarrier wait; lane 0 stores {total, wait0..wait3} per (CTA, warp) at kernel end (read back by dg_prof_read).
#ifdef DG_PROF
static __device__ long long dg_prof_buf[296][T3_W_LOAD + 1][5];
#define T3_WAIT(bar, par, id)            \
  do {                                   \
    const long long t0_ = clock64();     \
    tc::mbar_wait(bar, par);             \
    prof_[id] += clock64() - t0_;        \
  } while (0)
#else
#define T3_WAIT(bar, par, id) tc::mbar_wait(bar, par)
#endif
#ifdef DG_PROF
#define T3_TIMED(id, stmt)              \
  do {                                  \
    const long long t0_ = clock64();    \
    stmt;                               \
    prof_[id] += clock64() - t0_;       \
  } while (0)
#else
#define T3_TIMED(id, stmt) stmt
#endif

struct Tc3Params {
  StageParams s;
  const uint16_t *__restrict__ Bimg;   // [NSPLIT][NSTEP][3][2][NCH][8] bf16 operator panel image (host: build_tc3_image)
  const int *__restrict__ conn;        // [K][4] packed connectivity: (neighbour << 5 | face code) or -(bc tag)
  int nbatch;                          // end of the batch range this launch works on (all batches: ceil(K / EB))
  int bbeg;                            // first batch of the range (dg_stage_range; 0 otherwise)
  // epilogue TMA descriptors: 2-D views [K Nf rows][PT] of q_in, res and q_out | rhs with
  // boxes of CW nodes x 32 rows ([0]) and CW x (Nf EB - 96) rows ([1], the last row quadrant of an elastic batch)
  CUtensorMap tm_in[2], tm_res[2], tm_out[2];
  CUtensorMap tm_u;                    // q_in, boxes of 16 nodes x 128 rows, 64 B swizzle: the producers' field chunks (no tile)
  // MODE_AB3 (eq. (4)): boxes of CW / 2 nodes (three inputs per chunk share the staging of two): q_in, r^{m-1} (s.res),
  // r^{m-2} (s.hist2) in; r^m (s.rhs), q_out out
  CUtensorMap tm3_in[2], tm3_h1[2], tm3_h2[2], tm3_r0[2], tm3_out[2];
};

namespace tc {
// one lane of the (converged) warp; ptxas keeps the code under it on the uniform datapath
__device__ __forceinline__ bool elect_one() {
  uint32_t pred = 0;
  asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\t@P mov.u32 %0, 1;\n\t}\n" : "+r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void cp_async4(uint32_t dst, const float *src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(__cvta_generic_to_global(src)) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NWAIT>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(NWAIT) : "memory"); }
// 32 lanes x NCOL columns of TMEM -> NCOL registers per thread (NCOL = 16 or 32)
template <int NCOL>
__device__ __forceinline__ void tmem_ld(uint32_t taddr, uint32_t *v) {
  if constexpr (NCOL == 32) {
    tmem_ld32(taddr, v);
  } else if constexpr (NCOL == 8) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];\n\t"
        "tcgen05.wait::ld.sync.aligned;\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
        : "r"(taddr)
        : "memory");
  } else {
    static_assert(NCOL == 16, "8, 16 or 32 columns");
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n\t"
        "tcgen05.wait::ld.sync.aligned;\n"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
          "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
  }
}
// 2-D tiled TMA: global -> shared (completion on an mbarrier) and shared -> global (bulk async-group)
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *map, int x, int y, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
               "l"(map), "r"(x), "r"(y), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void tma_store_2d(const CUtensorMap *map, int x, int y, uint32_t src) {
  asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.tile.bulk_group [%0, {%1, %2}], [%3];" ::"l"(map), "r"(x), "r"(y), "r"(src)
               : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int NPEND>
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(NPEND) : "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void prefetch_l2(const void *src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(__cvta_generic_to_global(src)), "r"(bytes) : "memory");
}
}  // namespace tc

// ---- per-row pre-combination coefficients (rows a1 + a3), record in shared memory:
//      a_j = sum_i cf[j][i] * (u_src[i] - mean_i)
template <int MODEL>
__device__ __forceinline__ void row_coefficients_s(const float *g, int f, float cf[3][3], int src[3], int &nsrc) {
  float G[9];
#pragma unroll
  for (int i = 0; i < 9; ++i) G[i] = g[i];
#pragma unroll
  for (int j = 0; j < 3; ++j)
#pragma unroll
    for (int i = 0; i < 3; ++i) cf[j][i] = 0.f;
  src[0] = src[1] = src[2] = 0;
  if (MODEL == 0) {
    const float kap = g[9], irho = g[10];
    if (f == 0) {                   // eq. (5): r_p = -kappa sum_j D_j (sum_i g_ij v_i)
      nsrc = 3;
      src[0] = 1; src[1] = 2; src[2] = 3;
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int i = 0; i < 3; ++i) cf[j][i] = -kap * G[3 * i + j];
    } else {                        // eq. (6): r_vi = -(1/rho) sum_j g_ij D_j p
      nsrc = 1;
#pragma unroll
      for (int j = 0; j < 3; ++j) cf[j][0] = -irho * G[3 * (f - 1) + j];
    }
  } else {
    const float irho = g[9], lam = g[10], mu = g[11];
    nsrc = 3;
    if (f < 3) {                    // r_vi = (1/rho) sum_j D_j (sum_m g_mj sigma_im)
      const int row[3][3] = {{3, 6, 7}, {6, 4, 8}, {7, 8, 5}};
#pragma unroll
      for (int m = 0; m < 3; ++m) src[m] = row[f][m];
#pragma unroll
      for (int j = 0; j < 3; ++j)
#pragma unroll
        for (int m = 0; m < 3; ++m) cf[j][m] = irho * G[3 * m + j];
    } else {                        // PAPER.md:158 (reading Q6): lambda delta_ab div v + mu (d_b v_a + d_a v_b)
      src[0] = 0; src[1] = 1; src[2] = 2;
      const int a = f < 6 ? f - 3 : (f == 8 ? 1 : 0);
      const int bb = f < 6 ? f - 3 : (f == 6 ? 1 : 2);
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        if (f < 6) {
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
}

// ---- the kernel ------------------------------------------------------------------------------------
template <int MODEL, int N, int MODE>
__global__ void __launch_bounds__(T3_THREADS, 1) tc3_stage_kernel(const __grid_constant__ Tc3Params P) {
  using C = T3<MODEL, N>;
  constexpr int NP = C::NP, PT = C::PT, NFP = C::NFP, NFACE = C::NFACE, NF = C::NF, NGEO = C::NGEO, EB = C::EB, NCH = C::NCH;
  constexpr int NA = C::NA, NB = C::NB, NFL = C::NFL, NQ = C::NQ;
  constexpr bool TILE = C::TILE;
  const StageParams &p = P.s;

  extern __shared__ unsigned char smem_raw[];
  // 1024-byte aligned base (swizzled TMA boxes).  Pointer arithmetic on the __shared__ array, not an integer round trip:
  // the compiler then knows the address space and emits LDS / STS with 32-bit addresses instead of generic LD / ST
  unsigned char *sm = smem_raw + ((1024u - (tc::smem_u32(smem_raw) & 1023u)) & 1023u);
  unsigned char *sB = sm + C::OFF_B;                               // [NB][3][2][NCH][8] bf16
  float *s_flux = reinterpret_cast<float *>(sm + C::OFF_FLUX);     // [NFL][128][FLS] penalty-term chunks
  float *s_scr = reinterpret_cast<float *>(sm + C::OFF_SCR);       // epilogue staging (see the epilogue)
  unsigned char *s_u = sm + C::OFF_U;                              // [NU][128 rows][16] field chunks, 64 B swizzle
  unsigned char *s_slot = sm + C::OFF_SLOT;                        // [NQ] { field tile | geo | conn }
  uint64_t *bars = reinterpret_cast<uint64_t *>(sm + C::OFF_BAR);
  uint32_t *s_tmem = reinterpret_cast<uint32_t *>(bars + C::NBAR);

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int hid = C::NSPLIT == 1 ? 0 : (int)(blockIdx.x % C::NSPLIT);       // which half of the output nodes
  const int worker = (int)(blockIdx.x / C::NSPLIT), nworkers = (int)(gridDim.x / C::NSPLIT);
  const uint32_t bar0 = tc::smem_u32(bars);
  auto fullA = [&](int t) { return bar0 + 8u * t; };
  auto emptyA = [&](int t) { return bar0 + 8u * (NA + t); };
  auto fullB = [&](int t) { return bar0 + 8u * (2 * NA + t); };
  auto emptyB = [&](int t) { return bar0 + 8u * (2 * NA + NB + t); };
  auto flFull = [&](int t) { return bar0 + 8u * (2 * NA + 2 * NB + t); };
  auto flEmpty = [&](int t) { return bar0 + 8u * (2 * NA + 2 * NB + NFL + t); };
  const uint32_t barX = bar0 + 8u * (2 * NA + 2 * NB + 2 * NFL);
  auto accFull = [&](int t) { return barX + 8u * t; };
  auto accEmpty = [&](int t) { return barX + 8u * (2 + t); };
  auto qFull = [&](int t) { return barX + 8u * (4 + t); };
  auto qEmpty = [&](int t) { return barX + 8u * (6 + t); };
  auto epiFull = [&](int w, int t) { return barX + 8u * (8 + 3 * w + t); };
  auto uFull = [&](int t) { return barX + 8u * (20 + t); };
  auto uEmpty = [&](int t) { return barX + 8u * (20 + T3_NU + t); };

  if (warp == T3_W_MMA) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(tc::smem_u32(s_tmem)), "n"(512) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  if (tid == 0) {
    for (int t = 0; t < NA; ++t) { tc::mbar_init(fullA(t), 8); tc::mbar_init(emptyA(t), 1); }
    for (int t = 0; t < NB; ++t) { tc::mbar_init(fullB(t), 1); tc::mbar_init(emptyB(t), 1); }
    for (int t = 0; t < NFL; ++t) { tc::mbar_init(flFull(t), T3_FLUXW); tc::mbar_init(flEmpty(t), 8); }
    for (int t = 0; t < 2; ++t) {
      tc::mbar_init(accFull(t), 1); tc::mbar_init(accEmpty(t), 4);
      tc::mbar_init(qFull(t), 1); tc::mbar_init(qEmpty(t), 8 + T3_FLUXW);
    }
    for (int w = 0; w < 4; ++w)
      for (int t = 0; t < 3; ++t) tc::mbar_init(epiFull(w, t), 1);
    for (int t = 0; t < T3_NU; ++t) { tc::mbar_init(uFull(t), 1); tc::mbar_init(uEmpty(t), 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tm = *s_tmem;
#ifdef DG_PROF
  long long prof_[4] = {0, 0, 0, 0};
  const long long prof_t0 = clock64();
#endif

  if (warp < 4) {
    // =================================================== epilogue: LSRK update (row a7)
    // Chunks of 32 rows x CW output nodes move as 2-D TMA boxes: res / q in two chunks ahead (mbarrier per warp
    // and stage), results out through the same swizzled staging buffers (bulk async-group).  The update runs in
    // the TMEM-native layout (thread = row); the 128 B / 64 B swizzle keeps its float4 accesses conflict-free.
    // MODE_AB3 (the paper's update, eq. (4)) has three inputs per chunk (q, r^{m-1}, r^{m-2}) and two outputs (r^m, q): its
    // chunks are half as wide, so that three staging buffers per stage fit where the LSRK update keeps two.
    constexpr bool AB3 = MODE == MODE_AB3;
    constexpr int CW = AB3 ? C::CW / 2 : C::CW;
    constexpr int NBUF = AB3 ? 3 : 2;
    constexpr int LW = CW >= 16 ? 16 : 8;              // columns per TMEM load
    constexpr uint32_t BUFB = 32 * CW * 4;             // bytes of one staging buffer (aligned to 8 rows of it: the swizzle atom)
    constexpr int RLAST = C::NR - 96;                  // rows of the last quadrant (32 acoustic, 30 elastic)
    const int qd = warp;
    const int hmap = (qd == 3 && RLAST != 32) ? 1 : 0; // which box height
    const uint32_t boxbytes = (uint32_t)((hmap ? RLAST : 32) * CW * 4);
    constexpr int NES = C::NES;
    unsigned char *bufs = reinterpret_cast<unsigned char *>(s_scr) + warp * (NES * 2 * 32 * C::CW * 4);   // [stage][res | q (| r^{m-2})]
    const int n0 = hid * NCH;
    const int ncv = min(NCH, NP - n0);
    const bool need_res = MODE == MODE_STAGE && p.a != 0.f;
    const bool leader = tc::elect_one();               // the same lane issues and retires every TMA operation
    auto issue = [&](int stg, int b, int c0) {         // TMA loads of chunk (b, c0) into stage stg
      if (MODE != MODE_RHS && b < P.nbatch && leader) {
        const int row0 = b * EB * NF + qd * 32;
        const uint32_t dR = tc::smem_u32(bufs + (stg * NBUF) * BUFB), dQ = dR + BUFB;
        if (AB3) {
          tc::mbar_expect_tx(epiFull(warp, stg), 3 * boxbytes);
          tc::tma_load_2d(dQ, &P.tm3_in[hmap], n0 + c0, row0, epiFull(warp, stg));
          tc::tma_load_2d(dR, &P.tm3_h1[hmap], n0 + c0, row0, epiFull(warp, stg));
          tc::tma_load_2d(dQ + BUFB, &P.tm3_h2[hmap], n0 + c0, row0, epiFull(warp, stg));
        } else {
          tc::mbar_expect_tx(epiFull(warp, stg), need_res ? 2 * boxbytes : boxbytes);
          tc::tma_load_2d(dQ, &P.tm_in[hmap], n0 + c0, row0, epiFull(warp, stg));
          if (need_res) tc::tma_load_2d(dR, &P.tm_res[hmap], n0 + c0, row0, epiFull(warp, stg));
        }
      }
    };
    auto advance = [&](int &b, int &c0) {
      c0 += CW;
      if (c0 >= ncv) { c0 = 0; b += nworkers; }
    };
    int ab = P.bbeg + worker, ac0 = 0;                 // the chunk two ahead of the current one
    issue(0, ab, ac0);
    advance(ab, ac0);
    issue(1, ab, ac0);
    advance(ab, ac0);
    int it = -1, stg = 0, astg = 2 % NES, set = 0;     // stage of the current chunk / of the chunk two ahead
    uint32_t par = 0;                                  // phase bit per stage
    for (int b = P.bbeg + worker, c0 = 0; b < P.nbatch; advance(b, c0), stg = (stg + 1 == NES ? 0 : stg + 1)) {
      if (c0 == 0) {
        ++it;
        set = C::NSETS == 2 ? (it & 1) : 0;
        T3_WAIT(accFull(set), (C::NSETS == 2 ? (it >> 1) : it) & 1, 0);
        tc::tc_fence_after();
      }
      const uint32_t t0 = tm + ((uint32_t)(qd * 32) << 16) + set * 2 * NCH + c0;
      float acc[CW];                     // main + small accumulator, summed 16 columns at a time (register pressure)
      {
#pragma unroll
        for (int h = 0; h < CW / LW; ++h) {
          uint32_t vm[LW], vs[LW];
          T3_TIMED(2, tc::tmem_ld<LW>(t0 + LW * h, vm); tc::tmem_ld<LW>(t0 + NCH + LW * h, vs));
#pragma unroll
          for (int j = 0; j < LW; j += 2) {
            const float2 sum = __fadd2_rn(make_float2(__uint_as_float(vm[j]), __uint_as_float(vm[j + 1])),
                                          make_float2(__uint_as_float(vs[j]), __uint_as_float(vs[j + 1])));
            acc[LW * h + j] = sum.x;
            acc[LW * h + j + 1] = sum.y;
          }
        }
      }
      if (c0 + CW >= ncv) {              // accumulators drained: the MMA warp may start the next batch on this set
        tc::tc_fence_before();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(accEmpty(set));
      }
      if (MODE != MODE_RHS) {
        T3_WAIT(epiFull(warp, stg), (par >> stg) & 1, 1);   // this chunk's boxes have landed
        par ^= 1u << stg;
      }
      unsigned char *bR = bufs + (stg * NBUF) * BUFB, *bQ = bR + BUFB;
      // swizzle: 16-byte chunk j4 of row `lane` sits at chunk j4 ^ f(lane) (128B: lane & 7, 64B: (lane >> 1) & 3, 32B: (lane >> 2) & 1)
      const int sw = CW == 32 ? (lane & 7) : (CW == 16 ? ((lane >> 1) & 3) : ((lane >> 2) & 1));
#pragma unroll
      for (int j4 = 0; j4 < CW / 4; ++j4) {
        const int off = lane * (CW * 4) + ((j4 ^ sw) << 4);
        float4 *pr = reinterpret_cast<float4 *>(bR + off), *pq = reinterpret_cast<float4 *>(bQ + off);
        float r[4];
#pragma unroll
        for (int t = 0; t < 4; ++t) r[t] = acc[4 * j4 + t];
        if (MODE == MODE_RHS) {
          *pr = make_float4(r[0], r[1], r[2], r[3]);
        } else if (AB3) {                // eq. (4): q += dt (23/12 r^m - 16/12 r^{m-1} + 5/12 r^{m-2}); dt, a, b carry the products
          const float4 H1 = *pr, Q = *pq, H2 = *reinterpret_cast<const float4 *>(bQ + BUFB + off);
          *pr = make_float4(r[0], r[1], r[2], r[3]);
          *pq = make_float4(fmaf(p.b, H2.x, fmaf(p.a, H1.x, fmaf(p.dt, r[0], Q.x))), fmaf(p.b, H2.y, fmaf(p.a, H1.y, fmaf(p.dt, r[1], Q.y))),
                            fmaf(p.b, H2.z, fmaf(p.a, H1.z, fmaf(p.dt, r[2], Q.z))), fmaf(p.b, H2.w, fmaf(p.a, H1.w, fmaf(p.dt, r[3], Q.w))));
        } else {                         // res <- a res + dt r; q <- q + b res, two values per instruction (FMUL2 / FFMA2)
          float4 R = make_float4(0.f, 0.f, 0.f, 0.f);
          if (need_res) R = *pr;
          const float4 Q = *pq;
          const float2 a2 = make_float2(p.a, p.a), b2 = make_float2(p.b, p.b), dt2 = make_float2(p.dt, p.dt);
          const float2 R0 = __ffma2_rn(a2, make_float2(R.x, R.y), __fmul2_rn(dt2, make_float2(r[0], r[1])));
          const float2 R1 = __ffma2_rn(a2, make_float2(R.z, R.w), __fmul2_rn(dt2, make_float2(r[2], r[3])));
          const float2 Q0 = __ffma2_rn(b2, R0, make_float2(Q.x, Q.y)), Q1 = __ffma2_rn(b2, R1, make_float2(Q.z, Q.w));
          *pr = make_float4(R0.x, R0.y, R1.x, R1.y);
          *pq = make_float4(Q0.x, Q0.y, Q1.x, Q1.y);
        }
      }
      tc::fence_proxy_async();           // generic-proxy writes -> visible to the TMA store
      __syncwarp();
      if (leader) {
        const int row0 = b * EB * NF + qd * 32;
        if (MODE == MODE_RHS) {
          tc::tma_store_2d(&P.tm_out[hmap], n0 + c0, row0, tc::smem_u32(bR));
        } else if (AB3) {
          tc::tma_store_2d(&P.tm3_r0[hmap], n0 + c0, row0, tc::smem_u32(bR));
          tc::tma_store_2d(&P.tm3_out[hmap], n0 + c0, row0, tc::smem_u32(bQ));
        } else {
          tc::tma_store_2d(&P.tm_res[hmap], n0 + c0, row0, tc::smem_u32(bR));
          tc::tma_store_2d(&P.tm_out[hmap], n0 + c0, row0, tc::smem_u32(bQ));
        }
        tc::bulk_commit();
        tc::bulk_wait_read<NES - 2>();   // the stores of the stage refilled next have read their staging buffers
      }
      __syncwarp();
      issue(astg, ab, ac0);
      astg = astg + 1 == NES ? 0 : astg + 1;
      advance(ab, ac0);
    }
    if (leader) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  } else if (warp < 12) {
    // =================================================== producers: rows a1 + a3, BF16x3 split, tcgen05.st
    const int pw = warp - 4, qd = pw & 3, half = pw >> 2;
    const int r = qd * 32 + lane;                      // row = (element e, field f)
    const int e = r / NF, f = r - e * NF;
    const uint32_t trow = tm + ((uint32_t)(qd * 32) << 16) + C::ABASE + 4 * half;
    int slot = 0;
    uint32_t phase = 0;
    // One k-step of this row -> TMEM.  The completion of the tcgen05.st (wait::st, fence, arrive) of a k-step is
    // deferred until the pieces of the next one are computed, so that its latency overlaps that arithmetic.
    int pend = -1;                                     // A slot whose stores are in flight
    auto finish = [&]() {
      if (pend >= 0) {
        tc::tmem_st_wait();
        tc::tc_fence_before();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(fullA(pend));
        pend = -1;
      }
    };
    auto emit = [&](const float2 *a) {
      uint32_t p1[4], p2[4], p3[4];
#pragma unroll
      for (int t = 0; t < 4; ++t) tc::split3(a[t], p1[t], p2[t], p3[t]);
      finish();
      T3_WAIT(emptyA(slot), phase ^ 1, 0);
      tc::tc_fence_after();
      const uint32_t ta = trow + slot * T3_ASTRIDE;
      tc::tmem_st4(ta, p1[0], p1[1], p1[2], p1[3]);
      tc::tmem_st4(ta + 8, p2[0], p2[1], p2[2], p2[3]);
      tc::tmem_st4(ta + 16, p3[0], p3[1], p3[2], p3[3]);
      pend = slot;
      if (++slot == NA) { slot = 0; phase ^= 1; }
    };
    int it = 0, fc = 0, uc = 0;
    for (int b = P.bbeg + worker; b < P.nbatch; b += nworkers, ++it) {
      const int k0 = b * EB;
      const int nvalid = min(EB, p.K - k0);
      const bool valid = r < C::NR && e < nvalid;
      const int qs = it % NQ, quse = it / NQ;
      T3_WAIT(qFull(qs), quse & 1, 1);
      const unsigned char *sl = s_slot + qs * C::SLOT;
      const float *s_geo = reinterpret_cast<const float *>(sl + (TILE ? C::TILE_SLOT : 0));
      const float *qb = TILE ? reinterpret_cast<const float *>(sl) : p.q_in + (size_t)k0 * NF * PT;
      auto ldq = [&](const float *x) { return TILE ? *x : __ldg(x); };
      float cf[3][3];
      int src[3] = {0, 0, 0}, nsrc = 0;
      if (valid) {
        row_coefficients_s<MODEL>(s_geo + e * NGEO, f, cf, src, nsrc);
      } else {
#pragma unroll
        for (int j = 0; j < 3; ++j)
#pragma unroll
          for (int i = 0; i < 3; ++i) cf[j][i] = 0.f;
      }
      const float *sp[3];
      float mean[3];
#pragma unroll
      for (int i = 0; i < 3; ++i) {
        sp[i] = qb + (e * NF + src[i]) * PT;
        // mean of the four vertex values: D_j 1 = 0, so the shift is exact and removes the cancellation
        mean[i] = (valid && i < nsrc) ? 0.25f * ((ldq(sp[i]) + ldq(sp[i] + N)) + (ldq(sp[i] + C::NFP - 1) + ldq(sp[i] + NP - 1))) : 0.f;
      }
      // (packed FP32 arithmetic on register pairs from here on: FADD2 / FMUL2 / FFMA2)
      auto shifted = [&](const float4 &v, int i, float2 &lo, float2 &hi) {
        const float2 nm = make_float2(-mean[i], -mean[i]);
        lo = __fadd2_rn(make_float2(v.x, v.y), nm);
        hi = __fadd2_rn(make_float2(v.z, v.w), nm);
      };
      auto load_u = [&](int g, float2 (&u)[3][4]) {
        const int m0 = 16 * g + 8 * half;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          if (valid && i < nsrc && m0 < NP) {     // float4 reads: rows are 16-byte aligned (pitch PT), pad columns are zero
#pragma unroll
            for (int h4 = 0; h4 < 2; ++h4) {
              if (m0 + 4 * h4 < NP) {
                const float4 v = TILE ? *reinterpret_cast<const float4 *>(sp[i] + m0 + 4 * h4)
                                      : __ldg(reinterpret_cast<const float4 *>(sp[i] + m0 + 4 * h4));
                shifted(v, i, u[i][2 * h4], u[i][2 * h4 + 1]);
              } else {
                u[i][2 * h4] = u[i][2 * h4 + 1] = make_float2(0.f, 0.f);
              }
            }
          } else {
#pragma unroll
            for (int t = 0; t < 4; ++t) u[i][t] = make_float2(0.f, 0.f);
          }
        }
      };
      // without a tile the loader streams the fields as chunks of 16 nodes x 128 rows (64 B swizzle) through a ring
      auto load_u_ring = [&](int g, const unsigned char *ring, float2 (&u)[3][4]) {
        const int m0 = 16 * g + 8 * half;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
          if (valid && i < nsrc && m0 < NP) {
            const int rs = e * NF + src[i];
            const unsigned char *rowp = ring + rs * 64;
            const int sw = (rs >> 1) & 3;
#pragma unroll
            for (int h4 = 0; h4 < 2; ++h4) {
              if (m0 + 4 * h4 < NP) {
                const float4 v = *reinterpret_cast<const float4 *>(rowp + (((2 * half + h4) ^ sw) << 4));
                shifted(v, i, u[i][2 * h4], u[i][2 * h4 + 1]);
              } else {
                u[i][2 * h4] = u[i][2 * h4 + 1] = make_float2(0.f, 0.f);
              }
            }
          } else {
#pragma unroll
            for (int t = 0; t < 4; ++t) u[i][t] = make_float2(0.f, 0.f);
          }
        }
      };
#pragma unroll 1
      for (int g = 0; g < C::NG; ++g) {
        float2 u[3][4];
        if (TILE) {
          load_u(g, u);
        } else {
          const int us = uc % T3_NU, uuse = uc / T3_NU;
          ++uc;
          T3_WAIT(uFull(us), uuse & 1, 1);
          load_u_ring(g, s_u + us * T3_UCH, u);
          __syncwarp();
          if (lane == 0) tc::mbar_arrive(uEmpty(us));
        }
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          const float2 c0 = make_float2(cf[j][0], cf[j][0]), c1 = make_float2(cf[j][1], cf[j][1]), c2 = make_float2(cf[j][2], cf[j][2]);
          float2 a[4];
#pragma unroll
          for (int t = 0; t < 4; ++t) a[t] = __ffma2_rn(c2, u[2][t], __ffma2_rn(c1, u[1][t], __fmul2_rn(c0, u[0][t])));
          emit(a);
        }
      }
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(qEmpty(qs));      // this warp no longer reads the tile slot
#pragma unroll 1
      for (int h = 0; h < C::NH; ++h) {
        const int fs = fc % NFL, fuse = fc / NFL;
        constexpr int KPC = C::FCH / 16;                              // k-steps per flux chunk
        if (h % KPC == 0) T3_WAIT(flFull(fs), fuse & 1, 2);
        const float *fl = s_flux + fs * (128 * C::FLS) + r * C::FLS + 16 * (h % KPC) + 8 * half;
        float2 a[4];
        if (valid) {
          const float4 v0 = *reinterpret_cast<const float4 *>(fl);
          const float4 v1 = *reinterpret_cast<const float4 *>(fl + 4);
          // (columns beyond 4 Nfp hold zeros or finite penalty terms of an earlier chunk: the operator rows there are zero)
          a[0] = make_float2(v0.x, v0.y); a[1] = make_float2(v0.z, v0.w); a[2] = make_float2(v1.x, v1.y); a[3] = make_float2(v1.z, v1.w);
        } else {
#pragma unroll
          for (int t = 0; t < 4; ++t) a[t] = make_float2(0.f, 0.f);
        }
        if (h % KPC == KPC - 1 || h == C::NH - 1) {                   // done with the chunk
          __syncwarp();
          if (lane == 0) tc::mbar_arrive(flEmpty(fs));
          ++fc;
        }
        emit(a);
      }
      finish();                                        // the batch's last k-step must not wait for the next batch
    }
  } else if (warp < T3_W_OPS) {
    // =================================================== flux warps: rows a4 + a5, one 16-face-node chunk at a time
    const int ft = tid - 384;                           // 0 .. 32 T3_FLUXW - 1
    constexpr int TPT = C::TPT;
    // the ring starts out zeroed: slots are never fully overwritten (face-node padding, ragged batches), and what the
    // producers read there must at least be finite
    for (int x = ft; x < NFL * 128 * C::FLS; x += T3_FLUXW * 32) s_flux[x] = 0.f;
    unsigned short *s_nbrnode = reinterpret_cast<unsigned short *>(sm + C::OFF_TAB);   // [4][24][NFP]
    unsigned short *s_fmask = s_nbrnode + 96 * NFP;                                    // [4 NFP]
    for (int x = ft; x < 96 * NFP; x += T3_FLUXW * 32) s_nbrnode[x] = __ldg(p.nbrnode + x);
    for (int x = ft; x < NFACE; x += T3_FLUXW * 32) s_fmask[x] = __ldg(p.fmask + x);
    tc::named_bar_sync(1, T3_FLUXW * 32);
    int it = 0, fc = 0;
    for (int b = P.bbeg + worker; b < P.nbatch; b += nworkers, ++it) {
      const int k0 = b * EB;
      const int nvalid = min(EB, p.K - k0);
      const int qs = it % NQ, quse = it / NQ;
      T3_WAIT(qFull(qs), quse & 1, 0);
      const unsigned char *sl = s_slot + qs * C::SLOT;
      const float *s_geo = reinterpret_cast<const float *>(sl + (TILE ? C::TILE_SLOT : 0));
      const int *s_conn = reinterpret_cast<const int *>(s_geo + EB * NGEO);
      const float *s_q = reinterpret_cast<const float *>(sl);        // TILE only
      const float *gq = p.q_in + (size_t)k0 * NF * PT;                                 // the same values in global memory
#pragma unroll 1
      for (int h = 0; h < C::NHC; ++h, ++fc) {
        const int fs = fc % NFL, fuse = fc / NFL;
        if (p.pflux) {
          // interface-centric surface step (iface_kernels.cuh): the chunk's penalty terms are already in the face buffer
          // [K][Nf][4 Nfp]; rows (element, field) x FCH face nodes are copied into the ring slot, coalesced along the nodes
          constexpr int RPI = T3_FLUXW * 32 / C::FCH;                 // rows per pass
          const int jj = ft % C::FCH, j = C::FCH * h + jj;
          float v[(128 + RPI - 1) / RPI];
#pragma unroll
          for (int i = 0; i < (128 + RPI - 1) / RPI; ++i) {
            const int row = ft / C::FCH + RPI * i;
            v[i] = (j < NFACE && row < nvalid * NF) ? __ldg(p.pflux + ((size_t)k0 * NF + row) * NFACE + j) : 0.f;
          }
          T3_WAIT(flEmpty(fs), (fuse & 1) ^ 1, 1);
          float *fl = s_flux + fs * (128 * C::FLS);
#pragma unroll
          for (int i = 0; i < (128 + RPI - 1) / RPI; ++i) {
            const int row = ft / C::FCH + RPI * i;
            if (row < 128) fl[row * C::FLS + jj] = v[i];
          }
          __syncwarp();
          if (lane == 0) tc::mbar_arrive(flFull(fs));
          continue;
        }
        // ---- this thread's tasks of the chunk: one face node jj of the chunk, elements e0, e0 + EPI, ... (the face, the
        // interior node and the row of the neighbour-node table are the same for all of them)
        constexpr int EPI = T3_FLUXW * 32 / C::FCH;   // element stride between a thread's tasks
        const int jj = ft % C::FCH, e0 = ft / C::FCH, j = C::FCH * h + jj;
        const bool jvalid = j < NFACE;
        const int f = jvalid ? j / NFP : 0;
        const int nm = jvalid ? (int)s_fmask[j] : 0;
        const unsigned short *nbrow = s_nbrnode + (f * 24) * NFP + (j - f * NFP);
        // ---- gather the exterior traces (all loads in flight before the first use)
        float ext[TPT][NF];
        int cn[TPT];                                   // packed connectivity of the task's face; INT_MIN = no task
#pragma unroll
        for (int i = 0; i < TPT; ++i) {
          const int e = e0 + EPI * i;
          cn[i] = (int)0x80000000;
          if (jvalid && e < nvalid) {
            const int c4 = s_conn[e * 4 + f];
            cn[i] = c4;
            if (c4 >= 0) {
              const int nb = c4 >> 5;
              const int nn = nbrow[(c4 & 31) * NFP];
              const unsigned rel = (unsigned)(nb - k0);
              if (C::INBATCH && rel < (unsigned)nvalid) {    // neighbour inside the batch: its values are in the tile
                const float *qp = s_q + (rel * NF) * PT + nn;
#pragma unroll
                for (int c = 0; c < NF; ++c) ext[i][c] = qp[c * PT];
              } else {
                const float *qp = p.q_in + ((size_t)nb * NF) * PT + nn;
#pragma unroll
                for (int c = 0; c < NF; ++c) ext[i][c] = __ldg(qp + c * PT);
              }
            }
          }
        }
        T3_WAIT(flEmpty(fs), (fuse & 1) ^ 1, 1);    // producers have consumed the chunk that used this slot
        float *fl = s_flux + fs * (128 * C::FLS);
        // ---- penalty terms
#pragma unroll
        for (int i = 0; i < TPT; ++i) {
          if (cn[i] == (int)0x80000000) continue;
          const int e = e0 + EPI * i;
          const float *g = s_geo + e * NGEO;
          float um[NF];
          if (TILE) {
            const float *qm = s_q + (e * NF) * PT + nm;
#pragma unroll
            for (int c = 0; c < NF; ++c) um[c] = qm[c * PT];
          } else {
            const float *qm = gq + (e * NF) * PT + nm;
#pragma unroll
            for (int c = 0; c < NF; ++c) um[c] = __ldg(qm + c * PT);
          }
          float F[NF];
          if (MODEL == 0) {
            const float *fg = g + 12 + 5 * f;
            const float nx = fg[0], ny = fg[1], nz = fg[2];
            float dp, dvn;
            if (cn[i] >= 0) {
              dp = ext[i][0] - um[0];
              dvn = (ext[i][1] - um[1]) * nx + (ext[i][2] - um[2]) * ny + (ext[i][3] - um[3]) * nz;
            } else {
              acoustic_boundary_jump(cn[i], um[0], um[1] * nx + um[2] * ny + um[3] * nz, dp, dvn);
            }
            const float4 Pn = acoustic_penalty(g, fg, dp, dvn);
            F[0] = Pn.x; F[1] = Pn.y; F[2] = Pn.z; F[3] = Pn.w;
          } else {
            const float *fg = g + 16 + 8 * f;
            const float nx = fg[0], ny = fg[1], nz = fg[2];
            float Tmx, Tmy, Tmz;
            traction(um, nx, ny, nz, Tmx, Tmy, Tmz);
            float dv[3], dT[3];
            if (cn[i] >= 0) {
              float Tpx, Tpy, Tpz;
              traction(ext[i], nx, ny, nz, Tpx, Tpy, Tpz);
              dv[0] = ext[i][0] - um[0]; dv[1] = ext[i][1] - um[1]; dv[2] = ext[i][2] - um[2];
              dT[0] = Tpx - Tmx; dT[1] = Tpy - Tmy; dT[2] = Tpz - Tmz;
            } else {
              elastic_boundary_jump(cn[i], um, Tmx, Tmy, Tmz, nx, ny, nz, dv, dT);
            }
            elastic_penalty(g, fg, dv, dT, F);
          }
#pragma unroll
          for (int c = 0; c < NF; ++c) fl[(e * NF + c) * C::FLS + jj] = F[c];
        }
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(flFull(fs));
      }
      __syncwarp();
      if (lane == 0) tc::mbar_arrive(qEmpty(qs));
    }
  } else if (warp == T3_W_OPS) {
    // =================================================== operator stream (rows a2, a6): L2 -> shared-memory ring
    // (the whole warp runs the loop so that control flow stays uniform; one elected lane issues)
    const uint16_t *img = P.Bimg + (size_t)hid * C::NSTEP * (C::BSTAGE / 2);
    int slot = 0;
    uint32_t phase = 0;
    for (int b = P.bbeg + worker; b < P.nbatch; b += nworkers) {
      for (int st = 0; st < C::NSTEP; ++st) {
        T3_WAIT(emptyB(slot), phase ^ 1, 0);
        if (tc::elect_one()) {
          tc::mbar_expect_tx(fullB(slot), C::BSTAGE);
          tc::bulk_g2s(tc::smem_u32(sB + slot * C::BSTAGE), img + (size_t)st * (C::BSTAGE / 2), C::BSTAGE, fullB(slot));
        }
        __syncwarp();
        if (++slot == NB) { slot = 0; phase ^= 1; }
      }
    }
  } else if (warp == T3_W_MMA) {
    // =================================================== MMA issue: six BF16 MMAs per k-step
    constexpr uint32_t IDESC = tc::make_idesc_bf16(128, NCH);
    const uint64_t descB0 = tc::make_desc(tc::smem_u32(sB), NCH * 16, 128);
    int sa = 0, sb = 0, it = 0;
    uint32_t pa = 0, pb = 0;
    for (int b = P.bbeg + worker; b < P.nbatch; b += nworkers, ++it) {
      const int set = C::NSETS == 2 ? (it & 1) : 0, use = C::NSETS == 2 ? (it >> 1) : it;
      T3_WAIT(accEmpty(set), (use & 1) ^ 1, 0);
      tc::tc_fence_after();
      const uint32_t d0 = tm + set * 2 * NCH, d1 = d0 + NCH;
      for (int st = 0; st < C::NSTEP; ++st) {
        T3_WAIT(fullA(sa), pa, 1);
        T3_WAIT(fullB(sb), pb, 2);
        tc::tc_fence_after();
        if (tc::elect_one()) {
          const uint32_t a1 = tm + C::ABASE + sa * T3_ASTRIDE, a2 = a1 + 8, a3 = a1 + 16;
          const uint64_t b1 = descB0 + (uint64_t)(sb * 6 * NCH), b2 = b1 + 2 * NCH, b3 = b2 + 2 * NCH;
          const uint32_t acc = st > 0 ? 1u : 0u;
          tc::umma_bf16_ts(d1, a2, b1, IDESC, acc);    // cross terms, orders 2^-8 and 2^-16
          tc::umma_bf16_ts(d1, a1, b2, IDESC, 1u);
          tc::umma_bf16_ts(d1, a3, b1, IDESC, 1u);
          tc::umma_bf16_ts(d1, a2, b2, IDESC, 1u);
          tc::umma_bf16_ts(d1, a1, b3, IDESC, 1u);
          tc::umma_bf16_ts(d0, a1, b1, IDESC, acc);    // leading term
          tc::umma_commit(emptyA(sa));
          tc::umma_commit(emptyB(sb));
          if (st == C::NSTEP - 1) tc::umma_commit(accFull(set));
        }
        __syncwarp();
        if (++sa == NA) { sa = 0; pa ^= 1; }
        if (++sb == NB) { sb = 0; pb ^= 1; }
      }
    }
  } else {
    // =================================================== tile loader: fields, geometric records, connectivity
    int it = 0, uc = 0;
    for (int b = P.bbeg + worker; b < P.nbatch; b += nworkers, ++it) {
      const int k0 = b * EB;
      const int nvalid = min(EB, p.K - k0);
      const int qs = it % NQ, quse = it / NQ;
      T3_WAIT(qEmpty(qs), (quse & 1) ^ 1, 0);
      unsigned char *sl = s_slot + qs * C::SLOT;
      if (tc::elect_one()) {
        // rows are 16-byte aligned (pitch PT): the batch's fields are one aligned, contiguous run
        const float *src = p.q_in + (size_t)k0 * NF * PT;
        const uint32_t bq = (uint32_t)nvalid * NF * PT * 4u, bg = (uint32_t)nvalid * NGEO * 4u, bc = (uint32_t)nvalid * 16u;
        unsigned char *s_geo = sl + (TILE ? C::TILE_SLOT : 0);
        tc::mbar_expect_tx(qFull(qs), (TILE ? bq : 0u) + bg + bc);
        if (TILE) tc::bulk_g2s(tc::smem_u32(sl), src, bq, qFull(qs));
        tc::bulk_g2s(tc::smem_u32(s_geo), p.geo + (size_t)k0 * NGEO, bg, qFull(qs));
        tc::bulk_g2s(tc::smem_u32(s_geo + EB * NGEO * 4), P.conn + (size_t)k0 * 4, bc, qFull(qs));
        if (MODE == MODE_STAGE && p.a != 0.f) tc::prefetch_l2(p.res + (size_t)k0 * NF * PT, bq);
        if (MODE == MODE_AB3) {
          tc::prefetch_l2(p.res + (size_t)k0 * NF * PT, bq);
          tc::prefetch_l2(p.hist2 + (size_t)k0 * NF * PT, bq);
        }
      }
      __syncwarp();
      if (!TILE) {
        for (int g = 0; g < C::NG; ++g, ++uc) {          // the batch's fields, 16 nodes at a time
          const int us = uc % T3_NU, uuse = uc / T3_NU;
          T3_WAIT(uEmpty(us), (uuse & 1) ^ 1, 1);
          if (tc::elect_one()) {
            tc::mbar_expect_tx(uFull(us), T3_UCH);
            tc::tma_load_2d(tc::smem_u32(s_u + us * T3_UCH), &P.tm_u, 16 * g, k0 * NF, uFull(us));
          }
          __syncwarp();
        }
      }
    }
  }

#ifdef DG_PROF
  if (lane == 0 && blockIdx.x < 296) {
    long long *o = dg_prof_buf[blockIdx.x][warp];
    o[0] = clock64() - prof_t0;
    for (int i = 0; i < 4; ++i) o[1 + i] = prof_[i];
  }
#endif
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  if (warp == T3_W_MMA) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tm), "n"(512) : "memory");
  }
}

}  // namespace dgk
