/*
 * bemcub — C ABI of the B200 (sm_100a) library for the hot path of arXiv 1606.03743
 * (Glueck & Hilk, "Electric potential and field calculation of charged BEM triangles and
 * rectangles by Gaussian cubature").  Citations are to /root/reference/PAPER.md line numbers.
 *
 * What the library computes
 *   Every constant-sigma triangle / rectangle is replaced by the N weighted point charges of one
 *   of the paper's ten tabulated cubature rules (App. A/B, L283-386), q_i = w_i sigma A (L143),
 *   placed at Q_i by Eq. 3.3 (triangle, L109) or Eq. 3.2 (rectangle, L103).  Potential and field
 *   at a field point P are the direct sums of Eq. 4.1 (L139-143)
 *       Phi(P) = k sum_i q_i / |P-Q_i|,   E(P) = k sum_i q_i (P-Q_i) / |P-Q_i|^3,   k = 1/(4 pi eps0)
 *   over all points of all elements (L34, L202).  In distance-ratio-adaptive mode the rule of each
 *   (element, field point) pair is picked from DR = |P - Q_cen| / L (L66) by the limits of Sec. 4
 *   (L159), and pairs below the first limit use an exact closed-form integral of Eq. 2.1 (L62-64)
 *   instead.  The dense BEM collocation matrix (L34) is the same computation with unit sigma and
 *   the element centroids as field points, one entry per (row = field point, column = element).
 *
 * General conventions
 *   - Unless a parameter is marked HOST, every pointer is a DEVICE pointer owned by the caller
 *     (e.g. a PyTorch allocation) on the device given to bemcub_create.  The library never frees
 *     or keeps caller buffers; bemcub_set_elements copies what it needs into ctx-owned memory,
 *     and bemcub_eval copies sigma (see "sigma == NULL" there).
 *   - All work is enqueued on the CUDA stream given to bemcub_create (NULL = legacy default
 *     stream).  bemcub_eval / bemcub_assemble* are asynchronous: results are valid once the caller
 *     has synchronised that stream.  bemcub_set_elements, bemcub_solve, the *_host calls,
 *     bemcub_fp64_peak / bemcub_fp64_issue_sweep, bemcub_inner_loop_rate and bemcub_get_stats synchronise
 *     internally.  A call that has to grow ctx-owned scratch calls cudaFree / cudaMalloc (which
 *     synchronise the device); repeated calls of the same shapes do not.
 *   - Every function returns BEMCUB_OK (0) or a negative error code; nothing throws or longjmps
 *     across the ABI.  There is no CPU fallback: without a usable CUDA device bemcub_create fails.
 *   - SI units: lengths m, sigma C/m^2, Phi V, E V/m.  eps0 = 8.8541878128e-12 F/m (CODATA 2018;
 *     the paper prints no value), applied once after the summation.
 *   - A ctx is not thread-safe; use one ctx per host thread / stream.
 *
 * Element layout
 *   type[n]        uint8   BEMCUB_TRI or BEMCUB_RECT
 *   verts[n][3][3] double  triangle: vertices A, B, C (Eq. 3.3);
 *                          rectangle: corner P0, P1 = P0 + a u_x, P3 = P0 + b u_y (Eq. 3.2); the
 *                          fourth corner P0 + a u_x + b u_y is implied, Q_cen = P0 + (P1-P0)/2 + (P3-P0)/2
 *   sigma[n]       double  constant charge density of each element (L36, L62)
 *   L (L66) = (|AB|+|BC|+|CA|)/3 for a triangle, (a+b)/2 for a rectangle.
 */
#ifndef BEMCUB_H
#define BEMCUB_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bemcub_ctx bemcub_ctx; /* opaque; owns device scratch and the expanded points */

enum { BEMCUB_TRI = 0, BEMCUB_RECT = 1 };

/* rule levels: the triangle and rectangle rule of the same level are paired by degree (L125) */
enum {
  BEMCUB_RULE_ADAPTIVE = -1, /* per-pair choice by distance ratio (L159)                  */
  BEMCUB_RULE_L0 = 0,        /* Table A1 / B1: N = 4,        degree 3                      */
  BEMCUB_RULE_L1 = 1,        /* Table A2 / B2: N = 7,        degree 5                      */
  BEMCUB_RULE_L2 = 2,        /* Table A3 / B3: N = 12,       degree 7                      */
  BEMCUB_RULE_L3 = 3,        /* Table A4 / B4: N = 19 | 17,  degree 9                      */
  BEMCUB_RULE_L4 = 4,        /* Table A5 / B5: N = 33,       degree 12 | 13                */
  BEMCUB_LEVEL_ANALYTIC = 5  /* bit index of the analytic branch in use_levels_mask        */
};

/* methods of bemcub_eval_pairs besides the rule levels and BEMCUB_RULE_ADAPTIVE */
enum {
  BEMCUB_METHOD_ANALYTIC = 5,  /* the closed form of Eq. 2.1 at any distance                  */
  BEMCUB_METHOD_DUFFY_L0 = 8   /* + l (l = 0..4): rectangle rule of level l; on a triangle    */
                               /* through the Duffy map (L163-169), on a rectangle as it is    */
};

enum { BEMCUB_F64 = 0, BEMCUB_F32 = 1 };

enum {
  BEMCUB_OK = 0,
  BEMCUB_ERR_INVALID_ARG = -1,
  BEMCUB_ERR_DEGENERATE_ELEMENT = -2, /* an element with zero area / zero side            */
  BEMCUB_ERR_NOT_RECTANGLE = -3,      /* |e1.e2| > 1e-12 |e1||e2| for a BEMCUB_RECT        */
  BEMCUB_ERR_BAD_RULE = -4,
  BEMCUB_ERR_CUDA = -5,
  BEMCUB_ERR_NOMEM = -6,
  BEMCUB_ERR_NO_ELEMENTS = -7,        /* eval/assemble before a successful set_elements    */
  BEMCUB_ERR_NOT_CONVERGED = -8,      /* bemcub_solve: mat-vec limit reached (outputs valid) */
  BEMCUB_ERR_FIXED_SCRATCH = -9,      /* bemcub_eval_few_noalloc: more than its fixed scratch holds */
  BEMCUB_ERR_TOO_MANY_ELEMENTS = -10  /* bemcub_assemble*: mesh of more than 2^25 elements         */
};

/* Distance-ratio policy (Sec. 4).  dr[t][b], t = element type, are the UPPER distance-ratio
 * limits of the bands {analytic, N=33, N=19|17, N=12, N=7}; N=4 is used above dr[t][4].  A band
 * contains its lower limit (DR == limit belongs to the band above it): the decision is
 * "D^2 < (dr*L)^2" in double precision.  use_levels_mask: bit k (k = 0..4) enables rule level k,
 * bit 5 the analytic branch; a disabled choice moves to the next MORE accurate enabled one, or, if
 * there is none, to the most accurate enabled one (the paper's GPU integrator used N = 7/12/33 +
 * analytic only, L239).  allow_upgrade = 1 lets the library evaluate an (element, field-point
 * tile) with the most accurate rule any pair of the tile asks for, instead of choosing per pair;
 * results then differ from the per-pair policy only by the (smaller) truncation error of the
 * better rule.  Only cubature rules are upgraded to better cubature rules; the analytic branch
 * is always chosen pair by pair (its rounding error grows with the distance ratio, L44, so it
 * is no upgrade far away).  allow_upgrade = 0 reproduces the per-pair choice exactly. */
typedef struct {
  double dr[2][5];
  int32_t allow_upgrade;
  int32_t use_levels_mask;
} bemcub_policy;

/* Counters of the work enqueued by this ctx since creation / the last reset (host side). */
typedef struct {
  int64_t kernel_launches;     /* CUDA kernels of this library launched                    */
  int64_t point_interactions;  /* point-charge interactions of the last eval (fixed rule:   */
                               /* m * sum N; adaptive: counted on the device, valid after   */
                               /* the stream is synchronised and bemcub_get_stats is called)*/
  int64_t analytic_pairs;      /* (element, point) pairs sent to the analytic branch, ditto */
  int64_t last_eval_launches;  /* kernels launched by the most recent eval/assemble call    */
  int64_t kernel_cycles;       /* SM cycles and nanoseconds of the dominant kernel of the   */
  int64_t kernel_ns;           /* last eval/assemble call, read on the device (clock64 and  */
                               /* %globaltimer of one persistent CTA): cycles/ns = the SM   */
                               /* clock the kernel really ran at; 0 for calls with m <= 64  */
  int64_t fp64_instructions;   /* FP64 instructions per field point the interactions of the */
                               /* last eval/assemble executed: 18 (Phi+E), 12 (Phi), 28     */
                               /* (+gradient) per interaction; fewer where rules ran in      */
                               /* paired / median form (BEMCUB_PATH_PAIRED); 0 for FP32     */
  int64_t field_points_per_lane; /* R of the last bemcub_eval* call's kernel: the template      */
                               /* instantiation it ran (1, 2, 4; paired 1, 3, 5); tiles hold   */
                               /* 32 R field points; 0 for calls with m <= 64 (the tests use   */
                               /* it to know which instantiation a parity case reached)        */
} bemcub_stats;

/* device: CUDA device ordinal.  cuda_stream: a cudaStream_t cast to void* (NULL = default).    */
int bemcub_create(bemcub_ctx** out_ctx, int device, void* cuda_stream);
int bemcub_destroy(bemcub_ctx* ctx);

/* HOST struct.  want_field = BEMCUB_POLICY_POTENTIAL (0): the printed triangle-potential limits
 * 3/8/20/80/1500 (L159) for both element types; BEMCUB_POLICY_FIELD (1): limits for Phi and E together
 * ("slightly higher", L159): triangles 4/10/25/100/2000, rectangles 6/15/40/150/3000 (DESIGN.md
 * reading 7); BEMCUB_POLICY_FIELD_F32 (2): limits for calls with BEMCUB_F32 - the distance ratio from
 * which a rule's own field error is below the FP32 rounding floor of 1e-7 (triangles 2/2/3/6/25,
 * rectangles 2/3/4/8/30; Sec. 4 protocol, profiles/r2_accuracy_sweep.txt).
 * allow_upgrade = 1, use_levels_mask = 63.  Any other want_field: INVALID_ARG. */
enum { BEMCUB_POLICY_POTENTIAL = 0, BEMCUB_POLICY_FIELD = 1, BEMCUB_POLICY_FIELD_F32 = 2 };
int bemcub_default_policy(bemcub_policy* host_policy, int want_field);

/* Copies the mesh into the ctx and computes centroid, area and L of every element (Eq. 3.2/3.3,
 * L66).  Synchronises.  Errors: DEGENERATE_ELEMENT, NOT_RECTANGLE (the ctx then holds no mesh),
 * INVALID_ARG (n < 0, null pointers with n > 0, a type other than 0/1). */
int bemcub_set_elements(bemcub_ctx* ctx, int64_t n, const uint8_t* type, const double* verts);

/* Eq. 4.1 summed over all elements at m field points.
 *   sigma[n]; rule_id = BEMCUB_RULE_L0..L4 (fixed rule for every pair; no near-field switching: a
 *   field point that coincides with a Gaussian point gives IEEE inf/nan) or BEMCUB_RULE_ADAPTIVE
 *   (policy must be non-NULL; HOST pointer); field_pts[m][3]; out_phi[m]; out_E[m][3] or NULL.
 *   precision = BEMCUB_F64, or BEMCUB_F32: points, field points and the interaction arithmetic are
 *   FP32, sums of at most 128 terms are FP32 and those block sums are accumulated in FP64; the rule
 *   choice of BEMCUB_RULE_ADAPTIVE and the analytic branch stay FP64 (use the limits of
 *   BEMCUB_POLICY_FIELD_F32: the FP64 limits only buy points whose gain FP32 rounding hides);
 *   buffers keep their double type.
 * sigma == NULL: evaluate with the sigma of the previous call on this ctx that passed one (the ctx
 *   keeps a copy; INVALID_ARG if there is none).  Rule levels already expanded for that sigma are
 *   reused, so the preprocessing pass a1 is skipped - what a particle tracker wants, which asks
 *   for the field of the same charges at one point after the other (L32).  bemcub_set_elements
 *   drops the kept sigma; so does a bemcub_eval_linear call.
 * Calls with m <= 64 take a different route on the device: elements are spread over the lanes,
 *   every (element, point) pair gets its rule from its own distance ratio (allow_upgrade has no
 *   effect), the lanes' partial sums are combined with warp shuffles, and the Gaussian points
 *   are computed on the fly from the vertices (L218) - such a call has no preprocessing pass.
 * m = 0 is a no-op.  Asynchronous. */
int bemcub_eval(bemcub_ctx* ctx, const double* sigma, int rule_id, const bemcub_policy* host_policy,
                int64_t m, const double* field_pts, double* out_phi, double* out_E, int precision);

/* bemcub_eval for callers that are not allowed to allocate device memory: same arguments (FP64), same
 * kernel, same grid and therefore the same bits as a bemcub_eval call with m <= 64, but no cudaMalloc,
 * cudaFree or allocating library call is made - neither on this call nor on any later one.
 *   Who needs it.  A particle tracker (L32) asks for the field at one point after the other from inside
 *   its integration loop.  Such a loop often runs where allocating is forbidden or ruinous: in a host
 *   application that has handed all device memory to its own pool, next to other streams that a
 *   cudaMalloc would stall (it synchronises the whole device), or under a latency budget that one
 *   allocation would break.  bemcub_eval may allocate whenever a call is the first of its shape
 *   (partial sums) or brings a sigma (the ctx keeps a copy); this call never does.
 *   How.  The partial sums of the CTAs and the counters of the kernel live in one array that is part of
 *   the library image: 655,872 bytes (641 KB) on EVERY GPU on which this process has loaded the
 *   library, held until the process exits, whether or not this function is ever called.
 *   Limits.  1 <= m <= 64 field points per call (m = 0 is a no-op) on a device of at most 160 SMs;
 *   beyond either, BEMCUB_ERR_FIXED_SCRATCH and nothing is enqueued - split the points over several calls.
 *   sigma[n] must be passed (no NULL reuse): it is read in place, the ctx keeps nothing of this call, and
 *   the kept sigma / expanded points of earlier bemcub_eval calls stay as they were.  out_phi is required,
 *   out_E may be NULL.  The mesh is the one of bemcub_set_elements (which does allocate: set the mesh up
 *   before entering the region that must not).  bemcub_get_stats counts the launch but not its
 *   interactions; bemcub_last_path and the timing calls do not see it.
 *   First call on a device.  It asks the runtime for the array's address on that device (with the device
 *   made current) and remembers it for the process; make this first call during set-up, before any
 *   stream capture begins.
 *   Sharing.  There is ONE array per GPU for all contexts, streams and host threads of the process.  A call
 *   clears the counters it needs (stream-ordered) and overwrites the sums of the previous call, so calls
 *   that follow one another on one stream are safe; two calls that can be on the same GPU at the same time
 *   (different streams, or different ctxs on different streams) corrupt each other's results - serialise
 *   them.  Asynchronous, like bemcub_eval. */
int bemcub_eval_few_noalloc(bemcub_ctx* ctx, const double* sigma, int rule_id, const bemcub_policy* host_policy,
                            int64_t m, const double* field_pts, double* out_phi, double* out_E);

/* The single-element integrator (the paper's innermost layer, L193-196 item a; the unit of its
 * accuracy protocol, L68 and L149, Figs. 8-10): element k seen from field point k, k < npairs, NO
 * sum over elements.  Independent of the ctx mesh (bemcub_set_elements is not needed).
 *   type[npairs], verts[npairs][3][3] as in bemcub_set_elements; sigma[npairs] or NULL (unit density);
 *   field_pts[npairs][3]; out_phi[npairs]; out_E[npairs][3] or NULL.
 *   method = BEMCUB_RULE_L0..L4: Eq. 4.1 with the element's own rule of that level;
 *            BEMCUB_RULE_ADAPTIVE: rule or closed form by the pair's distance ratio (host_policy, HOST);
 *            BEMCUB_METHOD_ANALYTIC: the closed form (step a4) whatever the distance;
 *            BEMCUB_METHOD_DUFFY_L0 + l: the RECTANGLE rule of level l - on a triangle through the
 *            Duffy transformation Q = A + u[(B-A) + v(C-B)], u = (1+y)/2, v = (1+x)/2, weights (1+y) w
 *            (Sec. 4: "much larger errors": the mapped rule is exact for triangle polynomials
 *            of degree (D-1)/2 only), on a rectangle unchanged.
 *   precision = BEMCUB_F32: points and the interaction arithmetic in FP32 (closed form stays FP64).
 * A degenerate or non-rectangular element gives NaN in its own outputs (no error code: the call is
 * asynchronous and does not validate).  npairs = 0 is a no-op. */
int bemcub_eval_pairs(bemcub_ctx* ctx, int64_t npairs, const uint8_t* type, const double* verts, const double* sigma,
                      int method, const bemcub_policy* host_policy, const double* field_pts, double* out_phi,
                      double* out_E, int precision);

/* Field gradient from the same point charges (L273: derivatives of the field "can be easily
 * computed from the point charges"): out_G[m][6] = G_xx, G_yy, G_zz, G_xy, G_xz, G_yz with
 *     G_ab(P) = dE_a/dx_b = k sum_i q_i [ delta_ab / r_i^3 - 3 d_a d_b / r_i^5 ],  d = P - Q_i,
 * symmetric and traceless (G_zz is formed as -(G_xx + G_yy)); V/m^2.  Same arguments as
 * bemcub_eval (out_phi / out_E may be NULL; they are computed in the same pass), FP64 only.
 * Cubature rules only: in adaptive mode the policy must not enable the analytic branch
 * (use_levels_mask without bit 5, else INVALID_ARG) - the distance-ratio choice then ends at the
 * most accurate cubature rule.  28 FP64 instructions per point-charge interaction.  Asynchronous. */
int bemcub_eval_gradient(bemcub_ctx* ctx, const double* sigma, int rule_id, const bemcub_policy* host_policy,
                         int64_t m, const double* field_pts, double* out_phi, double* out_E, double* out_G);

/* Non-constant charge density (L275: "q_i = w_i A sigma(Q_i)"): sigma varies LINEARLY over each
 * element.  sigma_vertex[n][3] = its values at the three stored vertices (triangle A, B, C;
 * rectangle P0, P1, P3 - the implied fourth corner carries sigma_1 + sigma_3 - sigma_0).  Everything
 * else as bemcub_eval; only the charges of the expanded points change (preprocessing, a1).
 * Cubature rules only: in adaptive mode the policy must not enable the analytic branch (the
 * closed form is for constant sigma), else INVALID_ARG.  Asynchronous. */
int bemcub_eval_linear(bemcub_ctx* ctx, const double* sigma_vertex, int rule_id, const bemcub_policy* host_policy,
                       int64_t m, const double* field_pts, double* out_phi, double* out_E, int precision);

/* Dense collocation matrix (L34): out_matrix[i*ld + j] = k * Int_{element j} dS / |c_i - Q| (unit
 * sigma), c_i = centroid of element i, rule per pair by the policy (DR(i,j) uses L of element j;
 * the self term has D = 0 and is analytic).  Units V m^2 / C.  ld >= n.  The policy's
 * allow_upgrade is honoured per 32-row group of a 128-row tile.  Asynchronous.
 * bemcub_assemble_rows fills rows [row0, row0+nrows) only, into out_rows[(i-row0)*ld + j]
 * (row sharding across GPUs; sampling).
 * Limit: the mesh may have at most 2^25 = 33,554,432 elements (the fill kernel's queue of near pairs keeps
 * the column index in 25 bits) - also for a window of a few rows of a larger mesh; beyond it both calls
 * return BEMCUB_ERR_TOO_MANY_ELEMENTS and write nothing (the evaluation calls have no such limit). */
int bemcub_assemble(bemcub_ctx* ctx, const bemcub_policy* host_policy, double* out_matrix, int64_t ld);
int bemcub_assemble_rows(bemcub_ctx* ctx, const bemcub_policy* host_policy, int64_t row0, int64_t nrows,
                         double* out_rows, int64_t ld);

/* y[i] = sum_j matrix[i*ld + j] x[j], i, j < n: the product of a matrix filled by bemcub_assemble (or any
 * other n x n row-major FP64 matrix, ld >= n) with a vector - the potentials at the centroids for the
 * charge densities x (L34).  Bound by the HBM read of the matrix.  x and y must not overlap.  The sum of
 * a row is formed in a fixed order: results are reproducible.  Asynchronous. */
int bemcub_matvec(bemcub_ctx* ctx, const double* matrix, int64_t ld, const double* x, double* y);

/* Matrix-free solve of the collocation system (L34; "shell matrices ... not stored", L200):
 *     sum_j A_ij sigma_j = rhs_potential[i],  A as bemcub_assemble defines it (never formed),
 * by right-preconditioned (diagonal = analytic self terms) restarted GMRES(30); every mat-vec is
 * one potential-only adaptive evaluation at the n element centroids under `host_policy` (use
 * bemcub_default_policy(.., 0): the potential limits).  sigma[n]: initial guess on entry (zeros
 * are fine), solution on exit.  Stops when |rhs - A sigma|_2 <= rel_tol |rhs|_2 or after
 * max_matvecs mat-vecs - never more: the last one of the budget is kept for the residual of the
 * iterate returned (then BEMCUB_ERR_NOT_CONVERGED, with that iterate in sigma).
 * host_matvecs / host_rel_residual (HOST, may be NULL): mat-vecs used, true relative residual of sigma.
 * Synchronous.  The policy's allow_upgrade changes the operator only at the rules' truncation level. */
int bemcub_solve(bemcub_ctx* ctx, const bemcub_policy* host_policy, const double* rhs_potential, double* sigma,
                 double rel_tol, int max_matvecs, int* host_matvecs, double* host_rel_residual);

/* Lets bemcub_solve keep the matrix.  The paper's solver does not store it (L200) because its
 * meshes do not fit (1.5e6 elements: 18 TB); a B200 holds n up to about 1.4e5 (8 n^2 bytes of its 180 GB).
 * With max_matrix_bytes >= 8 n^2 a solve first fills the n x n matrix (as bemcub_assemble, under the
 * solve's policy) into ctx-owned memory - BEMCUB_ERR_NOMEM if that allocation fails - and every
 * mat-vec is a matrix-vector product read from HBM; larger meshes, and every mesh after
 * max_matrix_bytes = 0 (the default; it also frees the matrix), are solved matrix-free.  The two
 * operators differ at the rounding level of the entries only (same rules, same limits). */
int bemcub_solve_storage(bemcub_ctx* ctx, int64_t max_matrix_bytes);

/* Same as bemcub_set_elements / bemcub_eval with HOST buffers: copies the inputs to ctx-owned
 * device memory, runs, copies phi / E back and synchronises (the end-to-end path bench.py times). */
int bemcub_set_elements_host(bemcub_ctx* ctx, int64_t n, const uint8_t* host_type, const double* host_verts);
int bemcub_eval_host(bemcub_ctx* ctx, const double* host_sigma, int rule_id, const bemcub_policy* host_policy,
                     int64_t m, const double* host_field_pts, double* host_phi, double* host_E, int precision);

/* The tabulated rules (HOST outputs).  coords: triangle [N][3] barycentric (lambda_A, lambda_B,
 * lambda_C), rectangle [N][2] natural (x, y) in [-1,1]^2; w[N], sum w = 1 (Eq. 3.1). */
int bemcub_rule_info(int elem_type, int rule_id, int* npts, int* degree);
int bemcub_rule_points(int elem_type, int rule_id, double* host_coords, double* host_w);

/* Expanded point charges of the current mesh for one level, as the evaluation kernel reads them:
 * out_xyzq[n*stride][4] = (Q_i, q_i); stride = max N over the element types present; an element
 * with fewer points is padded with zero charges at its centroid.  sigma may be NULL (unit sigma).
 * Returns the stride in *out_stride.  Asynchronous. */
int bemcub_expand_points(bemcub_ctx* ctx, const double* sigma, int rule_id, double* out_xyzq, int* out_stride);

/* Centroid [n][3], area [n], L [n] of the current mesh (any pointer may be NULL).  Asynchronous. */
int bemcub_get_geometry(bemcub_ctx* ctx, double* out_cen, double* out_area, double* out_L);

/* Roofline denominator: the issue rate of the plain FP64 pipe.  bemcub_fp64_issue_sweep runs, for
 * about `seconds_per_variant` each, kernels that issue nothing but independent chains of FP64
 * instructions - mix 0: DFMA, 1: DADD, 2: DMUL, 3: the 8 DFMA : 6 DMUL : 4 DADD mix of Eq. 4.1, every
 * instruction reading at most two vector registers (the second source is a uniform register) - at 8,
 * 16 and 32 warps per SM.  Two further mixes document what costs issue cycles
 * and never win: 4: DFMA with three distinct, changing vector-register sources; 5: mix 0 with one
 * integer multiply-add after every second DFMA (its rate still counts the DFMAs only).
 * HOST outputs, index = mix * 3 + occupancy: host_rates[BEMCUB_PEAK_VARIANTS] in FP64
 * lane-instructions per second (warp instructions x 32), host_sm_mhz[BEMCUB_PEAK_VARIANTS] (may be
 * NULL) the SM clock during that launch (cycle counter / global timer).
 * bemcub_fp64_peak = the maximum of such a sweep lasting about `seconds` in total; flop/s = 2x (every
 * instruction counted as an FMA).  Both synchronise. */
#define BEMCUB_PEAK_VARIANTS 18
int bemcub_fp64_issue_sweep(bemcub_ctx* ctx, double seconds_per_variant, double* host_rates, double* host_sm_mhz);
int bemcub_fp64_peak(bemcub_ctx* ctx, double seconds, double* host_fp64_inst_per_s);

/* Second roofline reference: the evaluation kernels' own inner loop (Eq. 4.1: 18 FP64
 * instructions + one MUFU per point-charge interaction, 4 field points per lane, 12 warps per SM)
 * run for about `seconds` on data resident in shared memory, with no streaming, no rule selection
 * and no work queue.  Returns point-charge interactions per second: what the instruction mix of
 * the method itself allows on this GPU.  Synchronises. */
int bemcub_inner_loop_rate(bemcub_ctx* ctx, double seconds, double* host_interactions_per_s);

/* Device timing of the dominant kernel.  bemcub_set_timing(ctx, 1) makes every following
 * bemcub_eval / bemcub_assemble* call record CUDA events on the ctx stream: around the whole call
 * and around its dominant kernel (the evaluation kernel of a3, the fill kernel of a5).
 * bemcub_get_timing waits for the most recent such call to finish and returns both durations in
 * milliseconds (HOST outputs, either may be NULL); INVALID_ARG if no timed call has been made. */
int bemcub_set_timing(bemcub_ctx* ctx, int enable);
int bemcub_get_timing(bemcub_ctx* ctx, double* host_ms_total, double* host_ms_kernel);

/* Which kernel the last bemcub_eval* call of this ctx ran its field points through (HOST output): the
 * tests use it to know that a parity case exercised the path it was written for. */
enum {
  BEMCUB_PATH_NONE = 0,
  BEMCUB_PATH_FIXED = 1,     /* eval_fixed_kernel: one rule for every pair                               */
  BEMCUB_PATH_ADAPTIVE = 2,  /* eval_adaptive_kernel: rule per (element, tile) by distance ratio         */
  BEMCUB_PATH_PAIRED = 3,    /* eval_paired_kernel: the same with the rectangle rules' points in +- pairs */
                             /* and the 7-point triangle rule's points on the medians                    */
  BEMCUB_PATH_FEW = 4        /* eval_few_kernel: m <= 64, elements over the threads, rule per pair        */
};
int bemcub_last_path(bemcub_ctx* ctx, int* host_path);

/* HOST struct.  Synchronises the ctx stream when device counters of the last call are pending. */
int bemcub_get_stats(bemcub_ctx* ctx, bemcub_stats* host_stats);
int bemcub_reset_stats(bemcub_ctx* ctx);

const char* bemcub_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* BEMCUB_H */
