/* etac.h -- C ABI of the B200-native ETac tactile hot path (arxiv/paper_2604_20295).
 *
 * One call per RL step turns rigid contact into elastomer surface displacement for a batch of
 * E environments (Sec. III-A):
 *   S1  contact detection + penalty displacement of the ACTIVE nodes
 *   S2  decay-based linear propagation  u_i^j = exp(-alpha |p_j - p_i|) u^_j,
 *       Omega U_a                                                             (Eq. 1)
 *   S3  residual correction Phi (per-node MLP form of BASELINE.json)
 *   S4  mask M_p + combine  U_p = Omega U_a + Phi_p                           (Eq. 2)
 * alpha and the weights of Phi are inputs of etac_create.  Their calibration (Eq. 3) is
 * an offline loop of the caller; this library serves it with etac_backward (the gradients of one step) and
 * etac_update_params (writes a descent step back); the FEM data the paper calibrates on is not part of it.
 *
 * Conventions
 *   - All functions return etac_status; nothing throws; no global state.
 *   - "host" pointers are read during the call only (the ctx copies what it needs).
 *     "device" pointers must be CUDA device memory on the ctx's device, owned by the caller and
 *     kept alive until the stream reaches the end of the step.
 *   - etac_step only enqueues work on the given CUDA stream: no host synchronisation, no
 *     allocation, no host<->device copy of per-step data (so a step can be captured in a CUDA graph and
 *     replayed).  One in-flight stream per ctx;
 *     different ctxs are independent.  Each step depends only on its arguments (the model is
 *     quasi-static).
 *   - Units are the caller's: alpha is in 1/(unit of node_pos).  The synthetic workloads use mm.
 *   - Device-side data problems (NaN pose, non-unit quaternion) are not detected: the affected
 *     environment's output is unspecified, other environments are unaffected.
 *   - There is no CPU fallback: every entry point that computes needs a CUDA device of compute
 *     capability 10.x and fails with ETAC_ERR_UNSUPPORTED / ETAC_ERR_CUDA otherwise.
 */
#ifndef ETAC_H_
#define ETAC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ETAC_ABI_VERSION 7

typedef struct etac_ctx etac_ctx; /* opaque; owns every device allocation it makes */

typedef enum {
  ETAC_OK = 0,
  ETAC_ERR_INVALID_ARG = 1, /* NULL / out-of-range / inconsistent argument; ctx unchanged */
  ETAC_ERR_UNSUPPORTED = 2, /* valid request this build cannot serve (e.g. ETAC_PATH_DENSE on an fp32 context,
                               etac_backward with an ablation mode, a device that is not sm_100) */
  ETAC_ERR_ALLOC = 3,       /* host or device allocation failed */
  ETAC_ERR_CUDA = 4,        /* a CUDA call failed; etac_last_error() has the CUDA message */
  ETAC_ERR_CAPACITY = 5     /* n_envs > max_envs */
} etac_status;

/* Analytic indenters (north_star: "analytic indenter SDFs (sphere/box/capsule poses)").  The
 * signed distance is exact (1-Lipschitz), negative inside.  PAPER.md:L77 detects contact with
 * SDFs against object meshes; several indenters per environment are united by min. */
typedef enum { ETAC_IND_NONE = 0, ETAC_IND_SPHERE = 1, ETAC_IND_BOX = 2, ETAC_IND_CAPSULE = 3, ETAC_IND_GRID = 4 } etac_ind_type;

typedef struct {
  int32_t type;   /* etac_ind_type; NONE slots are skipped */
  float param[3]; /* sphere {r,-,-}; box {hx,hy,hz} half extents; capsule {r, half length along local z, -};
                     grid {grid id as a float,-,-}: a sampled SDF registered with etac_set_sdf_grid */
  float pose[7];  /* {px,py,pz, qx,qy,qz,qw}: unit quaternion, Isaac-Gym order; world frame */
  int32_t skip_patch1; /* self-contact (PAPER.md:L77 detects contact between the hand's own links too): the
                     other links' collision shapes are passed as indenters at their link poses, and the
                     shape of the link a patch is mounted on must not press on that patch: the patch with
                     index skip_patch1 - 1 ignores this indenter; 0 = no patch does */
} etac_indenter; /* 48 bytes */

enum { ETAC_KERNEL_EXP_L2 = 0 };                                  /* Eq. (1): exp(-alpha*|p_j-p_i|_2) */
enum { ETAC_RESID_NONE = 0, ETAC_RESID_PERNODE_MLP = 1, ETAC_RESID_POINTNET = 2 };
enum { ETAC_PREC_FP32 = 0, ETAC_PREC_BF16 = 1 };                  /* BF16: 16-bit tensor-core operands, fp32 accumulate */
enum { ETAC_ACTIVE_PASSTHROUGH = 0, ETAC_ACTIVE_PROPAGATE = 1 };  /* PASSTHROUGH: active rows keep u^ (mask M_p, L99) */
enum { ETAC_IN_INDENTERS = 0, ETAC_IN_PENETRATION = 1 };

typedef struct {
  uint32_t struct_size;        /* = sizeof(etac_model_desc); ABI check */
  int32_t n_nodes;             /* N >= 1 */
  const float* node_pos;       /* host [N x 3], undeformed positions P, patch-local frame */
  const float* node_normal;    /* host [N x 3], unit outward normals N */
  int32_t n_patches;           /* P >= 1 when patch_offset != NULL; ignored otherwise */
  const int32_t* patch_offset; /* host [P+1], 0 = off[0] < off[1] < ... < off[P] = N; nodes of a patch are
                                  contiguous and K is zero across patches.  NULL: patches are the connected
                                  components of the adjacency (must be contiguous index ranges), or one
                                  patch if there is no adjacency either. */
  const int32_t* adj_rowptr;   /* host [N+1] CSR mesh adjacency, optional (NULL) */
  const int32_t* adj_col;      /* host [adj_rowptr[N]] */
  int32_t kernel_type;         /* ETAC_KERNEL_EXP_L2 */
  int32_t n_alpha;             /* 1 or P */
  const float* alpha;          /* host [n_alpha], > 0 */
  int32_t resid_arch;          /* ETAC_RESID_* */
  int32_t resid_hidden;        /* 64 (only width built) */
  const float *W1, *b1, *W2, *b2, *W3, *b3; /* host, Linear-layer layout [out x in]:
                                  W1[64x9] (input order [u_lin(3), p(3), n(3)]) b1[64] W2[64x64] b2[64] W3[3x64] b3[3];
                                  may be NULL when resid_arch == ETAC_RESID_NONE */
  const float *E1, *e1, *E2, *e2, *G1, *g1, *D1, *d1, *D2, *d2; /* host, ETAC_RESID_POINTNET (the paper's form of
                                  Phi; widths are this library's reading, Fig. 3 is an image):
                                  per node f_i = silu(E2 silu(E1 [p,n,u^] + e1) + e2), E1[64x9] (input order
                                  [p(3), n(3), u^(3)], L93) e1[64] E2[64x64] e2[64]; per (env, patch)
                                  g = max_i f_i over all nodes of the patch, g' = silu(G1 g + g1), G1[64x64] g1[64];
                                  r_i = D2 silu(D1 [f_i; g'] + d1) + d2, D1[64x128] d1[64] D2[3x64] d2[3];
                                  may be NULL for the other forms */
  int32_t max_envs;            /* workspace sizing, >= 1 */
  int32_t max_indenters;       /* M >= 0: indenter slots per environment */
  int32_t precision;           /* ETAC_PREC_* */
  int32_t active_mode;         /* ETAC_ACTIVE_* */
  int32_t device;              /* CUDA ordinal */
} etac_model_desc;

/* Builds a context: validates, copies every host array, derives patches, builds the propagation
 * matrix K (Eq. 1) per patch on the device, stages the MLP weights, allocates the per-step
 * workspace for max_envs.  On failure *out is NULL.  The caller may free its arrays on return. */
etac_status etac_create(const etac_model_desc* desc, etac_ctx** out);

/* Frees everything the ctx owns after synchronising the device.  NULL is allowed. */
etac_status etac_destroy(etac_ctx* ctx);

typedef struct {
  uint32_t struct_size;               /* = sizeof(etac_step_args) */
  int32_t n_envs;                     /* 1..max_envs (0 is a no-op returning ETAC_OK) */
  int32_t input_mode;                 /* ETAC_IN_* */
  const etac_indenter* d_indenters;   /* device [E x max_indenters] (INDENTERS mode) */
  const float* d_patch_pose;          /* device [E x P x 7] {t, q} of every patch in the indenters' world frame,
                                         or NULL = identity */
  const float* d_penetration;         /* device [E x N] (PENETRATION mode): delta; negatives clamp to 0 */
  void* d_out;                        /* device displacement U, REQUIRED: element (e, i, c) at index
                                         e*out_env_stride + 3*i + c of an array of out_dtype; the 3N elements of
                                         every environment are fully overwritten, the gaps of a strided layout are
                                         not touched; patch-local frame (u^ = -delta * n with the create-time normal).
                                         Alignment: that of one element */
  float* d_penetration_out;           /* optional device [E x N]: delta */
  uint32_t* d_mask_out;               /* optional device [E x ceil(N/32)]: bit (i%32) of word i/32 = node i active */
  float* d_analytic_out;              /* optional device [E x N x 3]: unmasked K.U^ on ALL rows
                                         (the "linear decay only" term; test hook) */
  uint8_t* d_contact_out;             /* optional device [E x P]: 1 = some node of the patch is active; with one
                                         patch per link this is the link-contact vector S_cr of PAPER.md:L224 */
  int32_t* d_active_count_out;        /* optional device [E]: n_a = number of active nodes of the environment
                                         (contact ratio R_a = n_a / N) */
  int64_t out_env_stride;             /* elements between consecutive environments in d_out; 0 = 3N (packed),
                                         else >= 3N: U lands inside a wider per-env observation row (the n x 3
                                         tensor is the policy observation) */
  int32_t out_dtype;                  /* ETAC_OUT_*: fp32 (default) or bf16 (round to nearest even of the fp32 result) */
  int32_t reserved;                   /* 0 */
} etac_step_args;

/* Enqueues S1-S4 for n_envs environments on cuda_stream (a cudaStream_t; NULL = default stream).
 * Output for a patch none of whose nodes is in contact in that environment is exactly 0.
 * Reproducibility: repeated steps of the same inputs give the same bits, and an environment's result does not depend
 * on the other environments of the batch or on n_envs. */
etac_status etac_step(etac_ctx* ctx, void* cuda_stream, const etac_step_args* args);

/* Options / introspection. */
enum { ETAC_OPT_PATH = 1, ETAC_OPT_ABLATION = 2, ETAC_OPT_L2_GROUP_BYTES = 3 };
enum { ETAC_PATH_AUTO = 0, ETAC_PATH_DENSE = 1, ETAC_PATH_SPARSE = 2 };
/* DENSE : tcgen05 tensor-core contraction K_p . U^ (needs ETAC_PREC_BF16).  For patches of >= 2048 nodes (or when
 *         the U^ operand of a patch exceeds ETAC_OPT_L2_GROUP_BYTES) it is block-sparse: S1 records which 64-node
 *         k-blocks of a contacting (env, patch) hold an active node and sorts the environments of a patch by the
 *         position of their contact, and the contraction skips the k-blocks that no environment of a 32-env tile
 *         touches (Omega is (n-m) x m).  Skipped blocks contribute exact zeros: same result;
 * SPARSE: gather over the active nodes only (Omega U_a literally).  FP32 context: fp32 SIMT kernel,
 *         fp32 MLP.  BF16 context: bf16 K, fp32 u^ and accumulation, tensor-core MLP as in DENSE;
 *         selecting it allocates the active-node lists (16 bytes x max_envs x N), which is why the
 *         choice is made with etac_set_option and never inside etac_step;
 * AUTO  : DENSE for BF16 contexts, SPARSE for FP32 contexts.  (On a BF16 context the block-sparse DENSE form is
 *         faster than SPARSE at every contact fraction measured, 0.1 % .. 20 %, N = 256 .. 8192: BASELINE.md §4.) */
/* ETAC_OPT_ABLATION: the rows of Table II as run-time modes.  FULL (default):
 * U_p = M_p (Omega U_a + Phi_p) + active part.  RESIDUAL_ONLY: Phi_p without the linear term ("Residual
 * Network Only").  LINEAR_ONLY: Omega U_a without Phi_p ("Linear Decay Only"; same result as a context
 * created with ETAC_RESID_NONE).  NO_PROPAGATION: U = U^, i.e. the penalty displacement -delta*n of the
 * nodes in contact and 0 elsewhere (what a penalty-based simulator without propagation reports). */
/* ETAC_OPT_L2_GROUP_BYTES (default 40 MiB, >= 1): scheduling only, results do not depend on it.  The dense
 * contraction K_p . U^ walks a patch's work in groups of environment tiles whose U^ operand (6 bytes x nodes
 * of the patch per environment) fits this share of L2; when n_envs x 6 x (largest patch) is below it (and no patch
 * has 2048 nodes or more) the plain order is used (cfg 4). */
enum { ETAC_ABLATE_FULL = 0, ETAC_ABLATE_RESIDUAL_ONLY = 1, ETAC_ABLATE_LINEAR_ONLY = 2, ETAC_ABLATE_NO_PROPAGATION = 3 };
enum { ETAC_OUT_F32 = 0, ETAC_OUT_BF16 = 1 };
etac_status etac_set_option(etac_ctx* ctx, int32_t key, int64_t value);

enum {
  ETAC_INFO_N_NODES = 1,
  ETAC_INFO_N_PATCHES = 2,
  ETAC_INFO_MAX_ENVS = 3,
  ETAC_INFO_DEVICE_BYTES = 4,       /* bytes of device memory the ctx owns */
  ETAC_INFO_LAST_PATH = 5,          /* ETAC_PATH_* taken by the last step */
  ETAC_INFO_LAST_LAUNCHES = 6,      /* kernels launched by the last step */
  ETAC_INFO_LAST_CONTACT_PAIRS = 7, /* #(env,patch) pairs in contact in the last step; SYNCHRONISES the stream */
  ETAC_INFO_SM_COUNT = 8
};
etac_status etac_get_info(const etac_ctx* ctx, int32_t key, int64_t* value);

/* Sampled signed-distance field of an arbitrary object (PAPER.md:L77 queries SDFs against object
 * meshes; this is how such a field is handed over).  values[(iz*ny + iy)*nx + ix] (host, fp32) is the
 * SDF at origin + spacing*(ix, iy, iz) in the object's frame; an indenter of type ETAC_IND_GRID with
 * param[0] = grid_id places it with its pose.  The field at a point is the trilinear interpolation of
 * the samples at the point clamped to the grid's box plus the distance from the point to the box.
 * grid_id in [0, 8); nx, ny, nz >= 2; spacing > 0.  Copies the samples; replacing a grid synchronises
 * the device first.  Not to be called concurrently with etac_step on the same ctx. */
etac_status etac_set_sdf_grid(etac_ctx* ctx, int32_t grid_id, int32_t nx, int32_t ny, int32_t nz,
                              const float* origin, float spacing, const float* values);

/* Set-up helper for objects given as triangle meshes ("SDFs between nodes and object meshes"): samples
 * the signed distance field of a CLOSED, consistently oriented triangle mesh on the grid origin + spacing*(ix, iy, iz),
 * values_out[(iz*ny + iy)*nx + ix] -- the layout etac_set_sdf_grid takes, so that the object can be used as an
 * ETAC_IND_GRID indenter.  distance = min over the triangles of the distance to the triangle; negative where the
 * winding number of the surface around the point is >= 1/2 in magnitude (inside; either orientation).  Brute force on
 * `device` (one thread per grid point over all triangles, fp32), host pointers in and out (vertices [n_vertices x 3],
 * triangles [n_triangles x 3] vertex indices, origin [3]); allocates temporaries and synchronises: not for the step
 * loop.  ETAC_ERR_INVALID_ARG: NULL, fewer than 4 vertices / triangles, index out of range, non-finite vertex, grid
 * dimension < 2, spacing <= 0.  The message of a failure is etac_last_error(NULL). */
etac_status etac_mesh_to_sdf_grid(int32_t device, int32_t n_vertices, const float* vertices, int32_t n_triangles,
                                  const int32_t* triangles, int32_t nx, int32_t ny, int32_t nz, const float* origin,
                                  float spacing, float* values_out);

/* Message of the last failure on this ctx ("" if none); ctx-owned, valid until the next call.
 * With ctx == NULL returns the message of the last failed etac_create on this thread. */
const char* etac_last_error(const etac_ctx* ctx);

/* Host-only helper (no CUDA): connected components of a CSR adjacency as contiguous patches.
 * Writes off[0..*n_patches] (capacity cap entries).  ETAC_ERR_UNSUPPORTED if a component is not
 * a contiguous index range, ETAC_ERR_CAPACITY if cap is too small. */
etac_status etac_patches_from_adjacency(int32_t n_nodes, const int32_t* adj_rowptr, const int32_t* adj_col,
                                        int32_t* off, int32_t cap, int32_t* n_patches);

/* Backward pass for the calibration of Eq. (3) ("alpha and the residual network are
 * obtained by minimising || U_p - U_p* ||_2 by gradient descent"; Table I lists differentiability).
 * Given the upstream gradient G = dL/dU of one step (same inputs as etac_step), returns dL/dalpha and
 * dL/d(weights of the per-node residual MLP).  Rows that Eq. (2) overwrites with u^ (the active nodes,
 * ETAC_ACTIVE_PASSTHROUGH) and rows of contact-free (env, patch) pairs carry no gradient to them.  Optionally
 * also dL/d(penetration) and, chained through the SDF gradients, dL/d(indenter poses) and dL/d(patch poses) (see the
 * last two fields of etac_backward_args).  Arithmetic: fp32 on the fp32 copies of
 * K and the weights, whatever the context's precision; sums over environments use fp32 atomics, so
 * repeated calls agree to rounding, not bit for bit.  With ETAC_RESID_POINTNET (the network of PAPER.md:L91-L99,
 * whose input is [P, N, U^]) Phi does not depend on alpha, the weight gradients are those of its five layers and
 * dL/d(penetration) includes the path through the encoder input; the max-pool passes its gradient to the arg-max
 * row of every feature column.  Ablation modes other than FULL: ETAC_ERR_UNSUPPORTED.  Enqueues on cuda_stream, no host synchronisation. */
typedef struct {
  uint32_t struct_size;               /* = sizeof(etac_backward_args) */
  int32_t n_envs;                     /* 1..max_envs (0 is a no-op) */
  int32_t input_mode;                 /* ETAC_IN_*, as in etac_step_args */
  const etac_indenter* d_indenters;   /* device [E x max_indenters] */
  const float* d_patch_pose;          /* device [E x P x 7] or NULL */
  const float* d_penetration;         /* device [E x N] (PENETRATION mode) */
  const float* d_grad_out;            /* device [E x N x 3] fp32: dL/dU, REQUIRED */
  float* d_grad_alpha;                /* device [n_alpha] fp32, REQUIRED, overwritten: dL/dalpha (per patch if the
                                         context was created with n_alpha = P) */
  float* d_grad_weights;              /* device fp32, overwritten, or NULL; must be NULL for ETAC_RESID_NONE.
                                         ETAC_RESID_PERNODE_MLP: [4995] = dL/d W1[64x9] b1[64] W2[64x64] b2[64]
                                         W3[3x64] b3[3], in this order.  ETAC_RESID_POINTNET: [17411] = dL/d E1[64x9]
                                         e1[64] E2[64x64] e2[64] G1[64x64] g1[64] D1[64x128] d1[64] D2[3x64] d2[3] */
  float* d_grad_penetration;          /* device [E x N] fp32, overwritten, or NULL: dL/ddelta for the nodes in contact
                                         (u^ = -delta n, L77; the contact set is held fixed, 0 for the other nodes).
                                         The caller chains it to object / link poses through its SDF gradients, or
                                         asks for the two arrays below */
  /* dL/d(poses) (Table I: differentiability; delta comes from the SDFs of L77): dL/ddelta chained through the SDF
     gradient of the indenter that attains the union's min at each node in contact (contact set held fixed).  Both
     optional; ETAC_IN_INDENTERS mode only; need d_grad_penetration (read back by the kernel) and max_indenters <= 256.
     A row is (dL/dt[3], dL/dtheta[3]): t the pose's translation, theta a rotation applied on the LEFT in the world
     frame, R <- exp([theta]x) R (the torque about the body's own origin t, up to sign conventions of the caller).
     Where the SDF has no gradient -- a node on the shape's medial axis: the centre of a sphere, the axis segment of a
     capsule, a plane of equal distance to two faces inside a box, a cell face of a sampled grid -- the node's
     contribution has the direction rounding gives it (a set of measure zero in pose space).
     A struct_size that ends before these two fields is accepted (no pose gradients). */
  float* d_grad_indenter_pose;        /* device [E x max_indenters x 6] fp32, overwritten, or NULL; 0 for empty slots */
  float* d_grad_patch_pose;           /* device [E x P x 6] fp32, overwritten, or NULL; 0 if d_patch_pose is NULL */
} etac_backward_args;
#define ETAC_GRAD_WEIGHTS_LEN 4995
#define ETAC_GRAD_WEIGHTS_POINTNET_LEN 17411
etac_status etac_backward(etac_ctx* ctx, void* cuda_stream, const etac_backward_args* args);

/* Replaces the calibrated parameters of a context in place (one gradient-descent step of Eq. (3)):
 * alpha ([n_alpha], same n_alpha as at create; NULL = keep; K is rebuilt on the device) and / or the
 * weights of the context's residual network: the six arrays of the per-node MLP or the ten of the PointNet form (all
 * or none; layouts as in etac_model_desc).  Host pointers, copied.
 * Synchronises the device before and after; not to be called concurrently with etac_step /
 * etac_backward on the same ctx.  The result is the same as a context created with these parameters. */
typedef struct {
  uint32_t struct_size;   /* = sizeof(etac_params) */
  int32_t n_alpha;
  const float* alpha;
  const float *W1, *b1, *W2, *b2, *W3, *b3;
  const float *E1, *e1, *E2, *e2, *G1, *g1, *D1, *d1, *D2, *d2; /* ETAC_RESID_POINTNET contexts: all ten or none (layouts as
                                                                   in etac_model_desc); a struct_size that ends before E1
                                                                   is accepted (no PointNet arrays) */
} etac_params;
etac_status etac_update_params(etac_ctx* ctx, const etac_params* params);

/* Library ABI version (ETAC_ABI_VERSION the .so was built with). */
int32_t etac_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ETAC_H_ */
