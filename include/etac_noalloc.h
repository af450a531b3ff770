/* etac_noalloc.h -- one entry point of the ETac library that allocates NOTHING: no cudaMalloc / cudaFree, no context,
 * no allocating library routine.  For callers that cannot allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it).  Not part of the etac_create / etac_step path, which it leaves untouched.
 *
 * What it computes: the analytic propagation of ONE patch without a residual network,
 *     delta = max(penetration, 0), u^_j = -delta_j n_j for the active nodes (delta_j > 0, R5)
 *     passive row i :  U_i = sum_{j active} exp(-alpha ||p_j - p_i||_2) u^_j      (Eq. 1: Omega U_a)
 *     active row  i :  U_i = u^_i                                                 (mask M_p of Eq. 2)
 *     environment without an active node: all rows 0
 * i.e. what an ETAC_PREC_FP32 / ETAC_RESID_NONE context returns from etac_step in ETAC_IN_PENETRATION mode; fp32
 * arithmetic, the sum runs over the active nodes in node order.  K is evaluated on the fly (expf), not stored.
 *
 * Scratch: the compact per-environment lists of active nodes (index, u^) live in a file-scope
 * `static __device__ __align__(256)` array of ETAC_NOALLOC_MAX_ENTRIES entries of 16 bytes + ETAC_NOALLOC_MAX_ENVS
 * counters = 4 MiB + 16 KiB.  Every GPU that loads the library holds it until the process exits.  The limits:
 *     n_envs <= ETAC_NOALLOC_MAX_ENVS   and   n_envs * n_nodes <= ETAC_NOALLOC_MAX_ENTRIES
 * beyond them the call returns ETAC_ERR_CAPACITY and says so in err_msg; nothing is launched.
 * ALL calls on a device share the array and it keeps the last call's contents: a call overwrites the counters of
 * its environments before anything reads them (nothing has to start at zero) -- but two calls that OVERLAP on the
 * GPU (different streams, or graphs replayed concurrently) race on it.  Serialise them.
 *
 * Pointers are device pointers on the CURRENT device (cudaGetDevice), owned by the caller:
 *     d_pos, d_normal [n_nodes x 3] fp32 row-major, d_penetration [n_envs x n_nodes] fp32, d_out [n_envs x n_nodes x 3]
 *     fp32 (overwritten).  Enqueues two kernels on cuda_stream, no host synchronisation.
 * err_msg (host, may be NULL): receives a NUL-terminated message of at most err_cap bytes when the status is not ETAC_OK.
 * Status: ETAC_OK, ETAC_ERR_INVALID_ARG (NULL pointer, n < 0, alpha not finite or <= 0), ETAC_ERR_CAPACITY,
 * ETAC_ERR_CUDA.  n_envs == 0 or n_nodes == 0 is a no-op. */
#ifndef ETAC_NOALLOC_H_
#define ETAC_NOALLOC_H_
#include "etac.h"

#ifdef __cplusplus
extern "C" {
#endif

#define ETAC_NOALLOC_MAX_ENTRIES 262144 /* n_envs * n_nodes, 16 bytes each */
#define ETAC_NOALLOC_MAX_ENVS 4096

etac_status etac_propagate_noalloc(void* cuda_stream, int32_t n_envs, int32_t n_nodes, float alpha, const float* d_pos,
                                   const float* d_normal, const float* d_penetration, float* d_out, char* err_msg,
                                   int32_t err_cap);

#ifdef __cplusplus
}
#endif
#endif /* ETAC_NOALLOC_H_ */
