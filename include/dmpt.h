/*
 * dmpt.h - C ABI of the B200-native DNN-SP2-PT hot path (arXiv 2203.09621).
 *
 * The library computes, for a symmetric (already orthogonalised) Hamiltonian H0,
 * a symmetric perturbation H1 and an occupation count N_occ,
 *
 *     D0 = theta(mu I - H0),  Tr D0 = N_occ                       PAPER.md:72 (Eq. 5), 81
 *     D1 = d theta(mu I - (H0 + lambda H1)) / d lambda at 0        PAPER.md:164 (Eq. 20), 352 (Eq. 49)
 *
 * by the deep-layer recursion of Algorithms 1-3: per layer
 *     X0 = S0^2,  X1 = S0 S1 + S1 S0                               PAPER.md:497-499, Eqs. 25-26
 *     S0 <- sigma X0 + (1 - sigma) S0,  S1 <- sigma X1 + (1 - sigma) S1     Eqs. 23, 25
 * with every product taken in the dual half-precision representation A ~ A_hi + A_lo (both fp16),
 * A.B ~ A_hi.B_hi + A_hi.B_lo + A_lo.B_hi, fp32 accumulation, sigma_n
 * chosen by the trace criterion and both parameter-free stopping tests
 * (Eq. 78) evaluated on the device.
 *
 * Conventions
 *   - All matrices are row-major fp32 with a leading dimension in ELEMENTS (they are symmetric,
 *     so row-major == column-major).  "d_" arguments are DEVICE pointers, "h_" arguments HOST
 *     pointers.  The library never frees caller memory and allocates no device memory itself:
 *     the caller provides one workspace of dmpt_workspace_bytes() bytes (256-byte aligned).
 *   - Every kernel is enqueued on the cudaStream_t given to dmpt_create(); dmpt_run() returns
 *     after that stream has drained (it polls a pinned flag between chunks of layers; there is no
 *     host round trip per layer).
 *   - All functions return 0 on success or a negative DMPT_E* code; dmpt_strerror() describes it.
 *     There is no CPU fallback: without a CUDA device every compute call fails with DMPT_ECUDA.
 */
#ifndef DMPT_H
#define DMPT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DMPT_OK            0
#define DMPT_EINVAL       -1   /* null pointer, n <= 0, n_occ outside (0, n), ld < n, order not 0..3  */
#define DMPT_ESTATE       -2   /* dmpt_run before dmpt_set_hamiltonian                                */
#define DMPT_ECUDA        -3   /* CUDA error (text via dmpt_strerror / dmpt_last_cuda_error)          */
#define DMPT_EDEGENERATE  -4   /* eps_max - eps_min not positive and finite                           */
#define DMPT_ENOCONV      -5   /* max_layers reached; outputs hold the last iterate                   */
#define DMPT_ENUMERIC     -6   /* NaN/Inf in the scalar state, or fp16 overflow of a scaled iterate   */
#define DMPT_EWORKSPACE   -7   /* workspace too small or misaligned                                   */
#define DMPT_ELIMIT       -8   /* size beyond a compiled-in limit (DMPT_NOALLOC_MAX_N)                */

typedef struct dmpt_ctx dmpt_ctx;

typedef struct dmpt_options {
    int max_layers;    /* cap on the while loop of Algorithm 1 (the paper has none); default 200       */
    int order;         /* 1: D0, D1.  2: also D2 (Eq. 25 third line).  3: also D3 (Eq. 26 at  */
                       /* k = 3; results through dmpt_run_orders).  0: D0 only - the        */
                       /* ground-state DNN-SP2 recursion with Algorithm 2 as its stop (PAPER.md:176-186,   */
                       /* 515-519); pass NULL for every H1 / D1 argument                                  */
    int s0_shift;      /* a >= 0: S0 is split as hi = fp16(2^a S0), lo = fp16(2^a S0 - hi) and 2^-2a   */
                       /* is folded back in fp32 (exact).  0 = Eq. 13 verbatim.  -1 = default (14).    */
    int s1_autoscale;  /* 1 (default): the response iterates are split after an exact power-of-two     */
                       /* scale chosen on the device per layer from max|S1|; 0 = Eq. 43 verbatim.      */
    int bounds;        /* 0: Gershgorin discs of H0; 1: eps_min/eps_max below; 2: the     */
                       /* discs tightened on the device by lanczos_steps steps of the Lanczos recursion on   */
                       /* H0 (extreme Ritz values widened by the residual norm, intersected with the discs;   */
                       /* one HBM pass over H0 per step).  The bounds are inputs of the method                */
                       /* (PAPER.md:492): D0, D1 do not depend on them, the layer count does (about a third   */
                       /* fewer layers on dense random-orthogonal spectra).  dmpt_result::eps_min/max report  */
                       /* the pair that was used                                                              */
    double eps_min;    /* read only when bounds == 1                                                  */
    double eps_max;
    int wave_sync;     /* 1 (default): the CTAs of a layer launch re-align at every tile boundary so that   */
                       /* tiles in flight share operand panels through L2 (cooperative launch); 0: free run */
    int num_fields;    /* 1 (default; 0 reads as 1) .. 3 perturbations H1_a sharing H0, first order only:      */
                       /* D1_a for each in one run - S0^2 once per layer, S0.S1_a per field (the x, y, z       */
                       /* fields of the polarizability, Eq. 79).  Use the *_fields entry points.  */
    int epilogue_direct; /* 0 (default): the layer kernel's final epilogue goes through shared memory and TMA (old      */
                       /* iterate in, new iterate and its split out as full lines; the lower triangle of the fp32   */
                       /* iterates is restored when they leave the workspace); 1: every                             */
                       /* thread reads and writes its own row of the tile directly (round 1's path, kept for A/B     */
                       /* measurements; same arithmetic, bit-identical results)                                      */
    int lanczos_steps; /* bounds == 2: number of Lanczos steps, 1..64; 0 = default (20)                          */
    int no_pdl;        /* 1: do not chain the layer launches by programmatic dependent launch (A/B measurements;   */
                       /* results do not depend on it).  0 (default): launches that need no wave barrier are chained */
    int loop_graph;    /* 1: the layer loop runs on the device - ONE launch of a CUDA graph whose conditional WHILE   */
                       /* node has the launches of a layer as its body and the control step as its condition; the  */
                       /* host enqueues nothing per layer and looks at no flag (dmpt_run, dmpt_run_orders,          */
                       /* dmpt_run_fields; not the *_host calls, whose early read-back of D0 needs the host, nor    */
                       /* order 3).  0 (default): launches enqueued in chunks of 2-8 layers, two chunks ahead,      */
                       /* one pinned flag per chunk.  Same kernels, bit-identical results                           */
    int order0_narrow; /* order 0 only.  0 (default): the ground-state instantiation of the layer kernel, which stages  */
                       /* its two operands in k-blocks of 64 columns (128-byte rows: full stages, twice the bytes in   */
                       /* flight);                                                                                     */
                       /* 1: the general instantiation with 32-column k-blocks (A/B measurements; same k-steps in the  */
                       /* same order, bit-identical results)                                                           */
    int reserved[1];   /* must be 0                                                                   */
} dmpt_options;

typedef struct dmpt_result {
    int status;        /* same as the return code of dmpt_run                                         */
    int layers;        /* passes of the while loop of Algorithm 1; at order 0 the pass   */
                       /* on which Algorithm 2 fired is counted but its product is not formed            */
    int layers_d0;     /* layer at which the D0 test fired (Algorithm 2); 0 if it never did           */
    int layers_d1;     /* layer at which the D1 test fired (Algorithm 3); 0 if it never did           */
    int launches;      /* kernels this run launched (all of them this library's own)                  */
    int layers_d2;     /* order 2: layer at which the D2 test fired (R15); 0 otherwise            */
    int layers_d3;     /* order 3: layer at which the D3 test fired.  Multi-field runs: stop layer of field 3     */
                       /* (layers_d2: field 2, layers_d1: field 1)                                               */
    int reserved_i[1];
    double eps_min, eps_max;   /* spectral bounds used                                 */
    double fro_err0;           /* FroErr0 = ||S0 - S0^2||_F at the D0 stop layer; NaN at order 0 */
    double ms_total;           /* CUDA-event time of the whole run (bounds + transform + split + loop) */
    double ms_loop;            /* CUDA-event time of the layer loop alone ("time for main loop", Eq. 82)*/
    double ms_bounds;          /* a1: Gershgorin kernel, which also takes max|H1| (+ scalar set-up)      */
    double ms_transform;       /* a2 + a3 fused: S0, S1 and their first operand split (+ first decision) */
    double ms_split;           /* what follows it before the loop (order 2: S2_0 = 0 and its first scale) */
    double sm_clock_mhz;       /* SM clock of the layer loop, MHz: SM cycle counters over the device's nanosecond */
                               /* timer between the first and the last layer launch, all SMs; 0 if fewer than two  */
                               /* layers ran.  Under a power cap it lies below what nvidia-smi samples report.      */
    /* Per-layer records, entry n-1 for layer n.  Caller-allocated HOST arrays of max_layers
     * entries each, or NULL to skip.  Entries the run did not reach are left untouched. */
    int8_t *sigma;             /* sigma_n                                         */
    double *tr_s;              /* N_S = Tr S0_{n-1} entering layer n                                  */
    double *tr_x;              /* N_X = Tr (S0_{n-1})^2, evaluated as ||S0_{n-1}||_F^2 (R9) */
    double *id_err;            /* IdErr_n = N_S - N_X; NaN once S0 froze                              */
    double *fro_err1;          /* FroErr1_n; NaN before D0 converged                   */
    double *fro_err2;          /* FroErr2_n (order 2); NaN before D1 converged.  Multi-field: FroErr1 of field 2 */
    double *fro_err3;          /* order 3: FroErr3_n, NaN before D2 converged.  Multi-field: FroErr1 of field 3 */
} dmpt_result;

/* Defaults: max_layers 200, order 1, s0_shift -1, s1_autoscale 1, bounds 0, wave_sync 1, num_fields 1. */
void dmpt_default_options(dmpt_options *opt);

/* Bytes of device workspace dmpt_create() needs for matrices of size n at response order `order`
 * (0 on invalid arguments).  Layout is private; see DESIGN.md "HBM layout". */
size_t dmpt_workspace_bytes(int n, int order);

/* The same for a first-order context with num_fields (1..3) perturbations sharing H0. */
size_t dmpt_workspace_bytes_fields(int n, int num_fields);

/* Create a context for n x n problems.  `d_workspace` (device, >= dmpt_workspace_bytes(), 256-byte
 * aligned) stays owned by the caller and must outlive the context.  `cuda_stream` is a cudaStream_t
 * (NULL = the legacy default stream).  `opt` may be NULL for defaults. */
int dmpt_create(dmpt_ctx **ctx, int n, const dmpt_options *opt,
                void *d_workspace, size_t workspace_bytes, void *cuda_stream);

/* Register the problem: symmetric d_h0, d_h1 (device, fp32, leading dimension ld >= n) and n_occ in
 * (0, n).  The pointers are read by every later dmpt_run and must stay valid until then; symmetry
 * is a precondition and is not checked. */
int dmpt_set_hamiltonian(dmpt_ctx *ctx, const float *d_h0, const float *d_h1, int ld, int n_occ);

/* Run Algorithms 1-3 and write D0, D1 (and D2 when order == 2, else pass NULL) to device matrices
 * with leading dimension ld >= n.  `res` may be NULL.  On DMPT_ENOCONV the outputs hold the last
 * iterate.  Safe to call repeatedly.  Contexts of order 3 have one more output: use dmpt_run_orders
 * (dmpt_run and dmpt_run_host return DMPT_EINVAL for them). */
int dmpt_run(dmpt_ctx *ctx, float *d_d0, float *d_d1, float *d_d2, int ld, dmpt_result *res);

/* General response order (Eq. 26, 285 Eq. 40): the same run for a context of any
 * supported order m = 0..3.  d_d is a HOST array of m + 1 DEVICE matrices D0 .. D_m (leading dimension ld).  Per
 * layer the activation of order k is f^(k) = sum_j S^(j) S^(k-j); the terms with j > k/2 are the transposes of those
 * with j < k/2, so order k costs ceil(k/2) cross products M.Y + Y.M plus, for even k, one
 * square: order 3 adds  X3 = (S0 S3 + S3 S0) + (S1 S2 + S2 S1)  as one more launch per layer (twelve tensor-core
 * products per tile into two accumulators).  Stops are cascaded (R15): order k is tested with the
 * inequality of Algorithm 3 once order k-1 has converged.  H^(k) = 0 for k >= 2. */
int dmpt_run_orders(dmpt_ctx *ctx, float *const *d_d, int ld, dmpt_result *res);

/* Multi-field variants (contexts created with order == 1 and num_fields >= 1).
 * d_h1 / d_d1 are HOST arrays of num_fields DEVICE matrix pointers, all with leading dimension ld.
 * Every field runs Algorithm 3 on its own (its own stop layer, its own power-of-two scale); the run ends
 * when all have stopped.  Each D1_a is bit-identical to the single-field run of (H0, H1_a).  Per layer the
 * tensor work is 3 + 6 num_fields products per tile instead of 9 num_fields.  res->layers_d1/_d2/_d3 and
 * fro_err1/2/3 belong to fields 1/2/3. */
int dmpt_set_hamiltonian_fields(dmpt_ctx *ctx, const float *d_h0, const float *const *d_h1, int ld, int n_occ);
int dmpt_run_fields(dmpt_ctx *ctx, float *d_d0, float *const *d_d1, int ld, dmpt_result *res);
/* The multi-field run with HOST matrices (h_h1 / h_d1: host arrays of num_fields host matrix pointers; pinned memory
 * recommended): as dmpt_run_host, copies inside the call, D0 read back early. */
int dmpt_run_fields_host(dmpt_ctx *ctx, const float *h_h0, const float *const *h_h1, int ld_in, int n_occ,
                         float *h_d0, float *const *h_d1, int ld_out, dmpt_result *res);

/* The same call with HOST matrices (pinned memory recommended): copies H0, H1 to the device, runs,
 * and copies D0, D1 (D2) back.  ms_total then covers the copies too.  D0 is final as soon as Algorithm 2
 * fired, a few layers before the end: its read-back then starts on an internal copy stream and overlaps
 * the remaining layers (h_d0 must not be touched until the call returns, as for every output). */
int dmpt_run_host(dmpt_ctx *ctx, const float *h_h0, const float *h_h1, int ld_in, int n_occ,
                  float *h_d0, float *h_d1, float *h_d2, int ld_out, dmpt_result *res);

/* One dual-half product on its own (used by tests and micro-benchmarks of the layer kernel):
 * given symmetric device matrices S0, S1 (fp32, leading dimension ld), writes X0 = S0^2 and
 * X1 = S0 S1 + S1 S0 through exactly the split + tcgen05 path a layer takes (sigma = +1, no
 * stopping test).  Uses the context's workspace; invalidates nothing the caller owns. */
int dmpt_layer_products(dmpt_ctx *ctx, const float *d_s0, const float *d_s1, int ld,
                        float *d_x0, float *d_x1, int ld_out);

/* The order-2 product of one layer on its own (contexts created with order == 2 only; a9,
 * PAPER.md:195 Eq. 25 third line, 201 Eq. 26): given symmetric S0, S1, S2 writes
 * X2 = S0 S2 + S2 S0 + S1 S1, each of the three products in the dual half-precision form, through the
 * split + tcgen05 path of the order-2 pass of a layer (sigma = +1, no stopping test). */
int dmpt_layer_products2(dmpt_ctx *ctx, const float *d_s0, const float *d_s1, const float *d_s2, int ld,
                         float *d_x2, int ld_out);

/* The order-3 product of one layer on its own (contexts created with order == 3; Eq. 26 at k = 3):
 * X3 = S0 S3 + S3 S0 + S1 S2 + S2 S1 for symmetric S0..S3, through the split + tcgen05 path of the order-3 pass
 * (sigma = +1, no stopping test). */
int dmpt_layer_products3(dmpt_ctx *ctx, const float *d_s0, const float *d_s1, const float *d_s2, const float *d_s3,
                         int ld, float *d_x3, int ld_out);

/* A general product in the dual half-precision representation, on its own (the
 * congruence transforms either side of the hot path, H_orth = Z^T H Z and D = Z D_orth Z^T, PAPER.md:74-79,
 * A18, are two of these each): C = A.B^T = A_hi.B_hi^T + A_hi.B_lo^T + A_lo.B_hi^T for ANY n x n device
 * matrices A, B (fp32, leading dimension ld), fp32 accumulation promoted every 128 columns like the layer
 * products; each operand is split after its own power-of-two scale (max|.| into [8, 16)).  Contexts of
 * order >= 1.  C may alias A or B (both are copied into the workspace before C is written). */
int dmpt_product_nt(dmpt_ctx *ctx, const float *d_a, const float *d_b, int ld, float *d_c, int ld_out);

/* The congruence transforms of PAPER.md:74-79, 541 (Eq. 81), A17-A18, each two dmpt_product_nt products chained on
 * the device: transpose_z != 0: C = Z^T X Z (H_orth = Z^T H Z, Eq. 81);  transpose_z == 0: C = Z X Z^T (D = Z D_orth Z^T).
 * Z is any n x n device matrix, X a SYMMETRIC one (both fp32, leading dimension ld); where Z^T is needed as the row
 * operand it is transposed by the library's own copy kernel on the way into the workspace.  C may alias X or Z.
 * Contexts of order >= 1; uses the workspace's staging buffer (not concurrently with dmpt_run_host). */
int dmpt_congruence(dmpt_ctx *ctx, const float *d_z, const float *d_x, int ld, int transpose_z, float *d_c, int ld_out);

/* Finite-difference response from ground-state runs: the comparison the paper
 * draws in Fig. 5, built in as a validation / benchmark workload.  Contexts of order == 0.  For points == 2 (Eq. 83)
 *     D1 ~ [D(H0 + h H1) - D(H0 - h H1)] / 2h                                                  + O(h^2),
 * for points == 4 (Eq. 84)
 *     D1 ~ [-D(H0 + 2h H1) + 8 D(H0 + h H1) - 8 D(H0 - h H1) + D(H0 - 2h H1)] / 12h            + O(h^4),
 * every D(.) one run of the ground-state recursion (order 0) of this library on H0 + t H1 (formed on the device in
 * fp64, rounded once).  Cost in the paper's count: 2 products per layer and run, i.e. 4 (8) per layer
 * against 5 for the first-order recursion.  d_d1: device output (leading dimension ld_out); h_layers: host array of
 * `points` layer counts (may be NULL), in the order of the stencil terms above; *h_ms: CUDA-event time of all runs.
 * Returns the first non-zero status of the runs. */
int dmpt_fd_response(dmpt_ctx *ctx, const float *d_h0, const float *d_h1, int ld, int n_occ, double h, int points,
                     float *d_d1, int ld_out, int *h_layers, double *h_ms);

/* Inverse factor of a symmetric positive definite overlap matrix S (device, fp32, leading dimension ld):
 * Z with Z^T S Z = I by the third-order recursion of PAPER.md:693-703 (A19-A21),
 *     X_n = Z_n^T S Z_n,   Z_{n+1} = Z_n (1.875 I - 1.25 X_n + 0.375 X_n^2),   Z_0 = I / sqrt(eps_max(S)),
 * every product through dmpt_product_nt's kernel (four per iteration).  eps_max is the Gershgorin bound, which
 * the paper leaves open; all Z_n are then symmetric and the limit is S^(-1/2).  Stops when ||X_n - I||_F <= tol
 * or when it no longer decreases (the noise floor of the arithmetic, ~1e-5 sqrt(n)); DMPT_ENOCONV after max_iter
 * (<= 0: 30).  Writes Z to d_z (leading dimension ld_z), the iteration count and the last error (host).
 * Contexts of order >= 1; uses the workspace's staging buffers (not concurrently with dmpt_run_host). */
int dmpt_inverse_factor(dmpt_ctx *ctx, const float *d_s, int ld, float *d_z, int ld_z, int max_iter, double tol,
                        int *h_iters, double *h_err);

/* The three HBM-bound steps on their own (tests and micro-benchmarks; dmpt_run does not call these
 * entry points but launches the same kernels).  All run on the context's stream and return after it
 * drained.  Matrices are n x n (n of dmpt_create), row-major, leading dimensions in elements.
 *   a1  Gershgorin discs of d_h0 -> *h_eps_min, *h_eps_max (host).
 *   a2  S0 = (eps_max I - H0)/W, S1 = -H1/W, W = eps_max - eps_min (Eq. 34, 493), each
 *       element formed in fp64 and rounded once to fp32; *h_tr_s0 (host, may be NULL) = Tr S0.  (The kernel
 *       is the fused a2 + a3 kernel of dmpt_run: it also leaves the first operand split in the workspace.)
 *   a3  hi = fp16(2^shift x), lo = fp16(2^shift x - hi), round-to-nearest-even (Eq. 13);
 *       d_hi, d_lo are device fp16 (uint16_t bit patterns), leading dimension ld_out.  diag_half != 0
 *       splits x - I/2 instead (the form the order-0 operands take). */
int dmpt_spectral_bounds(dmpt_ctx *ctx, const float *d_h0, int ld, double *h_eps_min, double *h_eps_max);
int dmpt_initial_transform(dmpt_ctx *ctx, const float *d_h0, const float *d_h1, int ld,
                           double eps_min, double eps_max, float *d_s0, float *d_s1, int ld_out,
                           double *h_tr_s0);
int dmpt_split(dmpt_ctx *ctx, const float *d_x, int ld, int shift, int diag_half,
               uint16_t *d_hi, uint16_t *d_lo, int ld_out);

int dmpt_destroy(dmpt_ctx *ctx);

/* Order-parallel pair (Sec. III.C "parallelizing the matrix multiplications over
 * multiple GPU devices", 548-550): device0 computes f^(0) = S0^2 with the trace criterion and Algorithm 2, device1
 * computes f^(1) = S0 S1 + S1 S0 with Algorithm 3.  Information flows one way: per layer the fp16 operand pair of
 * S0_{n-1} (4 N^2 bytes) and a 40-byte decision record go from device0 to device1 by cudaMemcpyPeerAsync on a copy
 * stream, overlapping the products of both sides; there is no reduction and no collective.  After Algorithm 2 fired
 * the order-0 side is done and the order-1 side runs on alone (sigma flips).
 *   device0 == device1 is allowed (two streams of one GPU, device-local copies): the results - D0, D1, layer counts,
 *   per-layer records - are bit-identical to dmpt_run on the same inputs in both set-ups.
 * Workspaces: dmpt_pair_workspace_bytes(n, side) bytes on the respective device (side 0: order-0 side), 256-byte
 * aligned, caller-owned.  d_h0 and d_d0 live on device0, d_h1 and d_d1 on device1.  The pair owns its streams.
 * opt: as for dmpt_create with order 1 and one field (NULL for defaults).  The host keeps two layers of work queued
 * on either side and looks at one pinned flag per layer; it never waits for the layer it has just enqueued. */
typedef struct dmpt_pair dmpt_pair;
size_t dmpt_pair_workspace_bytes(int n, int side);
int dmpt_pair_create(dmpt_pair **pair, int n, const dmpt_options *opt,
                     int device0, void *d_workspace0, size_t workspace0_bytes,
                     int device1, void *d_workspace1, size_t workspace1_bytes);
int dmpt_pair_set_hamiltonian(dmpt_pair *pair, const float *d_h0, const float *d_h1, int ld, int n_occ);
int dmpt_pair_run(dmpt_pair *pair, float *d_d0, float *d_d1, int ld, dmpt_result *res);
int dmpt_pair_destroy(dmpt_pair *pair);
const char *dmpt_pair_last_cuda_error(const dmpt_pair *pair);

/* Step a1 for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc).  The Gershgorin discs of d_h0 (device, n x n, row-major, leading dimension ld >= n)
 * -> d_eps[0] = eps_min, d_eps[1] = eps_max (DEVICE, two doubles, caller-owned), in the arithmetic of
 * dmpt_spectral_bounds.  No context is needed; the call allocates nothing on the device or the host (no cudaMalloc,
 * cudaFree, cudaHostAlloc, no allocating library routine): its scratch - the disc ends of every row and one counter
 * - is a static device array of 256 + 16 DMPT_NOALLOC_MAX_N bytes (1 MiB) inside the library, held by every GPU
 * that loads libdmpt.so until the process exits.  The call enqueues one memset and one kernel on `cuda_stream`
 * (a cudaStream_t of the CURRENT device, which must also hold d_h0 and d_eps; NULL = the default stream) and returns
 * without waiting: d_eps is valid once the stream has reached that point.
 *   n > DMPT_NOALLOC_MAX_N -> DMPT_ELIMIT ("size beyond a compiled-in limit"), nothing enqueued; null pointers,
 *   n <= 0, ld < n -> DMPT_EINVAL; a failed launch -> DMPT_ECUDA.
 * All calls on one device share the scratch, which keeps the last call's contents: calls ordered on one stream (or
 * by events) are safe, calls that overlap on the GPU race on it and their results are undefined. */
#define DMPT_NOALLOC_MAX_N 65536
int dmpt_spectral_bounds_noalloc(const float *d_h0, int n, int ld, double *d_eps, void *cuda_stream);

const char *dmpt_strerror(int code);
/* Text of the last CUDA error seen by this context (empty string if none). */
const char *dmpt_last_cuda_error(const dmpt_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* DMPT_H */
