/* libdg -- C ABI of the B200 nodal-DG hot path (arxiv 1602.07997, PAPER.md).
 *
 * What the library computes (everything on one CUDA device, fp32):
 *   r_k(q)   the semi-discrete right-hand side of PAPER.md eq. (2)-(3):
 *            volume term   sum_ij g^vol_kij D_j f_jk   (eq. (5)-(6))
 *            surface term  sum_f g^sur_kf L_f p_kf     with the upwind penalty terms of
 *            PAPER.md:45-51 (acoustic) and PAPER.md:71-84 (elastic);
 *   the five-stage fourth-order low-storage Runge-Kutta update named by BASELINE.json
 *            res <- A_s res + dt r(q),  q <- q + B_s res   (replaces AB3, eq. (4));
 *   and, as the paper's own integrator, one AB3 step of eq. (4) (dg_ab3_step).
 *
 * Conventions:
 *   reference tetrahedron {r,s,t >= -1, r+s+t <= -1}; local vertices v1=(-1,-1,-1), v2=(1,-1,-1),
 *   v3=(-1,1,-1), v4=(-1,-1,1) in the order of `etov`; faces f0:(v1,v2,v3) f1:(v1,v2,v4)
 *   f2:(v2,v3,v4) f3:(v1,v3,v4).  `etov` may list an element's vertices in any order and with
 *   either orientation.  `bc[k][f]` always refers to face f of element k IN THE CALLER'S vertex
 *   order (the face opposite the caller's vertex 3, 2, 0, 1 for f = 0..3).  Internally an element
 *   with negative Jacobian has its last two vertices swapped at create time, which exchanges its
 *   faces 0 and 1; the library exchanges the two tags with them, so the caller never pre-swaps
 *   anything.  dg_node_coords, dg_geometry and dg_connectivity report the library's (swapped)
 *   vertex order: for such an element bctag / nrm / fscale columns 0 and 1 are the caller's 1 and 0.
 *   Nodes: Np=(N+1)(N+2)(N+3)/6 warp-and-blend nodes in lattice order, t slowest,
 *   then s, r fastest; dg_node_coords returns their physical coordinates.
 *   Field layout of q, rhs (DEVICE memory, caller-owned): [K][Nfields][Np] float, node index
 *   fastest (Table 1).  Acoustic fields (p,vx,vy,vz); elastic fields
 *   (vx,vy,vz,sxx,syy,szz,sxy,sxz,syz).
 *
 * Ownership: host arrays passed to dg_create are only read during the call.  The context owns
 * all device constants (operators, geometric factors, connectivity) and scratch (residual,
 * ping-pong state, AB3 history); dg_destroy frees them.  No device allocation after dg_create
 * (the tensor-core variant keeps a host-side cache of TMA descriptors for up to 64 caller
 * buffers, least recently used evicted; the library's own buffers are encoded at dg_create).
 * dg_rhs/dg_step/dg_run/dg_ab3_step are asynchronous on `cuda_stream` (a cudaStream_t passed as
 * void*, NULL = default stream; it must belong to the context's device) and never synchronise
 * the host.  Every entry point selects the context's device for the duration of the call and
 * restores the caller's current device before it returns (dg_create included).
 *
 * Errors: every int function returns 0 on success or a negative DG_ERR_* code; the message is
 * available from dg_last_error() (thread-local).  No exception crosses the boundary.
 */
#ifndef DG_H_
#define DG_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dg_ctx dg_ctx;

enum { DG_ACOUSTIC = 0, DG_ELASTIC = 1 };
/* tags for faces without a neighbour (reading Q9); SLIP is elastic-only (acoustic: = RIGID) */
enum { DG_BC_INTERIOR = 0, DG_BC_RIGID = 1, DG_BC_FREE = 2, DG_BC_SLIP = 3 };
enum {
  DG_OK = 0,
  DG_ERR_ARG = -1,      /* NULL pointer, N outside 1..10, unknown model, bad option            */
  DG_ERR_MESH = -2,     /* non-conforming mesh, degenerate element, untagged boundary face      */
  DG_ERR_MATERIAL = -3, /* rho<=0, c<=0, vs<=0 or vp <= vs*sqrt(4/3)                            */
  DG_ERR_CUDA = -4,     /* CUDA runtime failure, or a device entry point on a host-only context */
  DG_ERR_NOMEM = -5
};

typedef struct {              /* HOST pointers, borrowed during dg_create                        */
  int64_t nverts, K;
  const double *vxyz;         /* [nverts][3]                                                     */
  const int32_t *etov;        /* [K][4] vertex numbers, any orientation                          */
  const int8_t *bc;           /* [K][4] DG_BC_* for faces without neighbour; NULL => all RIGID   */
} dg_mesh;

typedef struct {              /* HOST, per element, fp64 (piecewise-constant media) */
  const double *rho;          /* [K]                                                             */
  const double *c_or_vp;      /* [K] acoustic c / elastic c_p                                    */
  const double *vs;           /* [K] elastic c_s (ignored for acoustic, may be NULL)             */
} dg_materials;

typedef struct {
  int device;                 /* CUDA device ordinal; -1 = host-only context (setup introspection,
                                 no device entry point works: they return DG_ERR_CUDA)           */
  int variant;                /* 0 = auto (1 for N = 1, 5 for N = 2, else 4); 1 = FP32 SIMT stage kernels (element per
                                 thread for acoustic N <= 2 / elastic N = 1, fused node per thread otherwise or when
                                 elems_per_thread / groups_per_cta is given);
                                 4 = pipelined warp-specialised tensor-core kernel (tcgen05, BF16x3 split, TMEM
                                 accumulators), every degree; needs 16-byte aligned q / rhs and K < 2^26;
                                 5 = FP32 SIMT row-per-thread kernel (thread = (element, field), operators in
                                 constant memory), N <= 3 (DG_ERR_ARG above); needs 16-byte aligned q / rhs.
                                 Any other value: DG_ERR_ARG                                           */
  int elems_per_thread;       /* 0 = auto; register blocking E of the SIMT kernel (1..8)         */
  int groups_per_cta;         /* 0 = auto; node groups G per CTA (CTA handles G*E elements)      */
  int max_ctas;               /* 0 = auto (one persistent CTA per SM); > 0 caps the grid of the
                                 tensor-core variant so that small test meshes give every CTA
                                 several batches (tests); < 0: DG_ERR_ARG                         */
  int surface;                /* 0 = element-centric (default): the stage kernel gathers the exterior traces and evaluates
                                 the penalty terms of its own elements; 1 = interface-centric (the surface kernel of the
                                 paper's SGEMM strategy): a separate kernel visits every interface once, one
                                 thread per face node computes the terms of both sides into a face buffer
                                 [K][Nfields][4 Nfp], and the stage kernel lifts from it (one more launch per evaluation) */
  int64_t owned_elements;     /* 0 = all; > 0: the first `owned_elements` elements of the mesh are this process's own, the
                                 rest are ghost copies of other processes' elements (dg_partition_*): every device entry
                                 point advances / evaluates the owned elements only; ghosts are read through the
                                 connectivity and filled by dg_halo_unpack                                          */
} dg_options;

/* Build a context: reference operators for degree N (1..10), geometric factors, connectivity,
 * material constants; uploads them and allocates scratch.  `opts` may be NULL (device 0, auto). */
int dg_create(dg_ctx **out, const dg_mesh *mesh, int N, int model, const dg_materials *mat,
              const dg_options *opts);
int dg_destroy(dg_ctx *ctx);

/* sizes */
int dg_num_fields(const dg_ctx *ctx);         /* 4 or 9                                          */
int dg_np(const dg_ctx *ctx);                 /* nodes per element                               */
int dg_nfp(const dg_ctx *ctx);                /* nodes per face                                  */
int64_t dg_num_elements(const dg_ctx *ctx);

/* physical node coordinates, HOST out [K][Np][3] */
int dg_node_coords(const dg_ctx *ctx, double *xyz_host);
/* dt = cfl / ((N+1)^2 max_k [c_max,k max_f g^sur_kf])   (reading Q10); <0 on error   */
double dg_stable_dt(const dg_ctx *ctx, double cfl);

/* r(q) -> d_rhs.  DEVICE pointers, [K][Nfields][Np] float each; d_q is not modified;
 * d_q == d_rhs is an error.                                                                     */
int dg_rhs(dg_ctx *ctx, const float *d_q, float *d_rhs, void *cuda_stream);
/* one LSRK(5,4) step in place on d_q (5 fused stage kernels + one device copy)                  */
int dg_step(dg_ctx *ctx, float *d_q, float dt, void *cuda_stream);
/* nsteps LSRK steps in place on d_q (5*nsteps fused stage kernels, one copy if that is odd)     */
int dg_run(dg_ctx *ctx, float *d_q, float dt, int nsteps, void *cuda_stream);
/* dg_step for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same LSRK(5,4) step (row a7 of the path fused into the five stage kernels, BASELINE.json north_star),
 * the same kernels, the same result as dg_step bit for bit -- but the work memory of the step (the residual, the
 * ping-pong copy of q and, where the tensor-core kernel keeps padded rows, the private padded state) lives in ONE
 * file-scope `static __device__` array of DG_STATIC_SCRATCH_BYTES inside the library instead of buffers owned by the
 * context.  The call performs no cudaMalloc / cudaFree and calls no allocating library routine: it enqueues one memset
 * of the part of the array it uses, the five stage kernels (plus two row re-pitch kernels for padded rows) and one
 * device copy on `cuda_stream`.  (dg_create, at set-up, does allocate the context's constants; it also resolves the
 * array's device address, once per device.)
 *   d_q     DEVICE, [K][Nfields][Np] float, 16-byte aligned, updated in place; caller-owned.
 *   limit   2 (3 with padded rows: tensor-core kernel at N = 4, 8, 10) arrays of K Nfields Np floats, each rounded up to
 *           256 bytes, must fit in DG_STATIC_SCRATCH_BYTES; beyond that the call returns DG_ERR_ARG with a message that
 *           names the size needed and the limit, and enqueues nothing.
 *   sharing every context, every stream and every call on a device shares the one array, and it keeps the last call's
 *           contents: each call clears what it uses first, so results never depend on earlier calls, but two calls that
 *           overlap on the GPU (different streams, or different host threads without ordering) RACE on it -- order
 *           them on one stream or with events.  The context's own residual (dg_stage, dg_run) is not touched.
 *   cost    every GPU on which the library's module is loaded holds the DG_STATIC_SCRATCH_BYTES until the process exits.
 * Errors: as dg_step; DG_ERR_CUDA if the array's address could not be resolved (cudaGetSymbolAddress).             */
#define DG_STATIC_SCRATCH_BYTES (32 * 1024 * 1024)
int dg_step_static(dg_ctx *ctx, float *d_q, float dt, void *cuda_stream);
/* ONE low-storage stage with explicit coefficients, out of place (the building block of dg_run, exposed for
 * per-stage control: sampled full-size parity checks, multi-rate drivers):
 *   res <- a res + dt r(q_in);  q_out <- q_in + b res     (res is the context's residual array; a = 0 ignores it).
 * d_q_in is not modified; d_q_in == d_q_out is an error (neighbours read the stage input).                     */
int dg_stage(dg_ctx *ctx, const float *d_q_in, float *d_q_out, float a, float b, float dt, void *cuda_stream);
/* ---- hooks for multi-rate (local) time stepping (elements advance with a step that fits
 * their own size and wave speed; the drivers of refs [16,17,33] are not part of this library).  A driver numbers the
 * elements level by level (dg_element_dt gives each element's own stable step), then advances one level at a time:
 * dg_stage_range is dg_stage restricted to the elements k_begin <= k < k_end -- q_out and the residual of every other
 * element are left untouched, exterior traces are read from d_q_in whatever range the neighbour is in (the driver
 * keeps / interpolates the coarse levels' states there: "trace buffering").  k_begin and k_end must be multiples of
 * dg_range_alignment() (k_end may also be K).  Not available where the library pads rows (DG_ERR_ARG).              */
int dg_element_dt(const dg_ctx *ctx, double cfl, double *dt_host /* [K] */);
int dg_range_alignment(const dg_ctx *ctx);
int dg_stage_range(dg_ctx *ctx, const float *d_q_in, float *d_q_out, float a, float b, float dt, int64_t k_begin,
                   int64_t k_end, void *cuda_stream);
/* The paper's own time integrator, third-order Adams-Bashforth (eq. (4)):
 *   q^{m+1} = q^m + dt (23/12 r^m - 16/12 r^{m-1} + 5/12 r^{m-2}),   one evaluation of r per step.
 * The context keeps r^{m-1}, r^{m-2} (R_-1, R_-2 of Table 1).  Steady state: ONE fused kernel per step
 * (r(q), the combination and the rotation of the history by pointer); d_q is updated in place (ping-pong inside, one
 * device copy per call if the number of steps is odd: prefer dg_ab3_run over repeated dg_ab3_step).  Start-up (DESIGN.md
 * reading Q21 -- the paper does not say how the first two steps are taken): while fewer than two earlier right-hand sides
 * are on record (after dg_create / dg_ab3_reset) a step is r(q) into the history plus one LSRK(5,4) step, which keeps the
 * third order.  dt must be the same from step to step (dg_ab3_reset when it changes).                               */
int dg_ab3_step(dg_ctx *ctx, float *d_q, float dt, void *cuda_stream);
int dg_ab3_run(dg_ctx *ctx, float *d_q, float dt, int nsteps, void *cuda_stream);
int dg_ab3_reset(dg_ctx *ctx, void *cuda_stream);

/* number of kernels/copies the last dg_rhs/dg_step/dg_run/dg_ab3_step call enqueued             */
int dg_last_launch_count(const dg_ctx *ctx);
/* name of the kernel variant chosen at create time, e.g. "simt_fused<acoustic,N=5,E=4,G=2>"     */
const char *dg_variant_name(const dg_ctx *ctx);

/* ---- host-side introspection (no device work; valid on host-only contexts too) -------------
 * reference operators as the device sees them, fp64 before rounding: Dr,Ds,Dt [Np][Np] row-major,
 * LIFT [Np][4Nfp] row-major, rst [Np][3], fmask [4][Nfp].  Any pointer may be NULL.             */
int dg_reference_operators(const dg_ctx *ctx, double *Dr, double *Ds, double *Dt, double *LIFT,
                           double *rst, int32_t *fmask);
/* per element geometric factors: G [K][3][3] (G[i][j] = d r_j / d x_i), J [K], nrm [K][4][3],
 * fscale [K][4]; connectivity as (element, volume node) of the exterior trace of every face
 * node: elemP, nodeP [K][4Nfp] (boundary faces: the element's own node), bctag [K][4].           */
int dg_geometry(const dg_ctx *ctx, double *G, double *J, double *nrm, double *fscale);
int dg_connectivity(const dg_ctx *ctx, int32_t *elemP, int32_t *nodeP, int8_t *bctag);

/* ---- multi-GPU: element partition and halo exchange (one process per GPU) ------------------
 * The element list is cut into `nranks` contiguous slabs.  dg_partition_create builds, for one rank, its local mesh =
 * its own elements followed by ghost copies of the elements across its cut faces (vertex numbers stay global: pass the
 * same vxyz to dg_create, with dg_options.owned_elements = dg_partition_num_owned), and per peer rank the lists of faces
 * (4 * local element + face, the library's face numbering) whose face-node values are sent (own elements) and received
 * (ghosts), in matching order on both sides.  Host only.  Before every stage:
 *   dg_halo_pack(send faces) -> exchange the buffers [nfaces][Nfields][Nfp] float (NCCL send/recv or peer copies; the
 *   caller's plumbing) -> dg_halo_unpack(recv faces) -> dg_stage.  Only face traces move: Nfields Nfp floats per cut face
 *   and direction.  d_faces are DEVICE copies of the lists; d_q is in the caller's layout [K][Nfields][Np].            */
typedef struct dg_part dg_part;
int dg_partition_create(dg_part **out, const dg_mesh *mesh, int nranks, int rank);
int dg_partition_destroy(dg_part *part);
int64_t dg_partition_num_owned(const dg_part *part);
int64_t dg_partition_num_ghost(const dg_part *part);
int dg_partition_global_ids(const dg_part *part, int64_t *ids /* [owned + ghost] */);
int dg_partition_local_mesh(const dg_part *part, int32_t *etov /* [owned + ghost][4] */, int8_t *bc /* [owned + ghost][4] */);
int dg_partition_num_peers(const dg_part *part);
int dg_partition_peer(const dg_part *part, int i, int *rank, int64_t *nsend, int64_t *nrecv);
int dg_partition_halo_faces(const dg_part *part, int i, int32_t *send_faces /* [nsend] */, int32_t *recv_faces /* [nrecv] */);
int dg_halo_pack(dg_ctx *ctx, const float *d_q, const int32_t *d_faces, int64_t nfaces, float *d_buf, void *cuda_stream);
int dg_halo_unpack(dg_ctx *ctx, float *d_q, const int32_t *d_faces, int64_t nfaces, const float *d_buf, void *cuda_stream);
int64_t dg_num_owned_elements(const dg_ctx *ctx);

const char *dg_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DG_H_ */
