/* nqs.h — C ABI of the B200-native local-energy hot path of arxiv 2208.05637
 * ("Scalable Neural Quantum States Architecture for Quantum Chemistry").
 *
 * What the library computes (citations are PAPER.md lines of /root/reference/PAPER.md):
 *
 *   l_theta(x) = sum_{p in S} alpha_p <x|P_p|x^p> f(x^p, theta) / f(x, theta)          (:152, Eq. 15)
 *   <x|P_p|x^p> = (-i)^r prod_{k: p_k in {2,3}} (-1)^{x_k},  r = #sigma_2 in P_p      (:158 Eq. 16, :192)
 *   x^p = x xor F^{1,2}_p                                                             (:128, Alg. 1 line 1)
 *   log f(x) = i phi(x) + 1/2 sum_i log pi_i(x_i | x_<i)                              (:96, Eq. 10)
 *
 * with pi_i the conditionals of a MADE (masked FC -> ReLU -> ... -> sigmoid, :84) and phi a dense
 * two-layer MLP on the first n-2 inputs with 4 outputs picked by the last two bits (:84-86, :91).
 *
 * Conventions.  Qubit j (0-based) <-> bit j%64 of word j/64 of a 2 x uint64 configuration; x_j = 1 is
 * |1> (occupied).  Pauli codes 0,1,2,3 = sigma_0..sigma_3 = I,X,Y,Z (:40 Eq. 1).  Per term:
 * f = positions holding X or Y (the paper's F^{1,2}), s = positions holding Y or Z (F^{2,3}).
 * n_qubits in [3, 128].  All "host" pointers are ordinary CPU memory, all "_dev" pointers are CUDA
 * device memory of the current device (e.g. torch tensor.data_ptr()); `cuda_stream` is a cudaStream_t
 * passed as void* (NULL = legacy default stream).
 *
 * Ownership.  Handles are created by the library and released only by the matching *_free.  Every
 * buffer passed in stays owned by the caller and is not referenced after the call returns
 * (compile/create copy what they need).
 *
 * Errors.  Every int-returning function returns NQS_OK (0) or a negative nqs_status; on error `*out`
 * handles are left untouched.  Nothing aborts, throws across the ABI or prints.  There is no CPU
 * fallback: compute entry points return NQS_ECUDA / NQS_EARCH when no sm_100 device is usable.
 */
#ifndef NQS_H_
#define NQS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nqs_ham  nqs_ham_t;    /* opaque: compiled Hamiltonian (host copy + device term tensors) */
typedef struct nqs_made nqs_made_t;   /* opaque: packed MADE + phase-MLP parameters (host + device)     */

enum nqs_status {
    NQS_OK           =  0,
    NQS_EINVAL       = -1,   /* NULL pointer, negative size, Pauli code > 3, bits >= n_qubits set, bad permutation */
    NQS_ERANGE       = -2,   /* n_qubits outside [3,128], hidden < 1 or > 1024, degrees outside [1, n-1], ...    */
    NQS_ENOMEM       = -3,   /* host or device allocation failed                                                 */
    NQS_ECUDA        = -4,   /* a CUDA runtime call or kernel launch failed (no device, ...)                      */
    NQS_EARCH        = -5,   /* device is not compute capability 10.x (the kernels are sm_100a only)             */
    NQS_EUNSUPPORTED = -6    /* the requested path cannot run this shape (e.g. NQS_PATH_TC on hidden > 512)       */
};

/* Which kernels evaluate the MADE chain.  Both are CUDA; neither touches the CPU.  Callers pass NQS_PATH_AUTO; the two
 * explicit values exist for the parity tests and the benchmark (the fp32 path is the GPU-side reference of the tensor-core
 * path and the only path for shapes the latter does not take) — there is one implementation per shape, not a dispatch
 * between backends.
 *  NQS_PATH_SIMT : fp32 FFMA on CUDA cores, every layer (any shape; the parity reference for the tensor-core path).
 *  NQS_PATH_TC   : tcgen05 tensor cores driven by CTA pairs (cta_group::2), fp16 operands / fp32 accumulation in
 *                  TMEM, fused gather of x xor f into the operand tile and log|psi| / phase / ratio / E_loc in the
 *                  epilogue.  Needs n_hidden_layers in {1, 2}, hidden in [1, 512] (padded inside the library to a
 *                  multiple of 128 with zero-weight units: the padded network is the same function, exactly) and
 *                  n_qubits in [3, 126]: the operand tile carries two constant columns for the hidden-layer biases,
 *                  so round16(n+2) <= 128 input columns; TMEM holds two 128-column accumulators + round16(n+4)
 *                  output columns + round16(n+2)/2 input columns <= 512 (three accumulators when n <= 76).  Other
 *                  shapes (n = 127, 128 included) return NQS_EUNSUPPORTED; NQS_PATH_AUTO then takes NQS_PATH_SIMT.
 *                  Precision: hidden (padded) >= 384 runs ONE fp16 pass (10-bit mantissa, the TF32 mantissa): every psi
 *                  ratio carries a relative error of a few 1e-4, so |dE_loc| is bounded by ~8e-3 sum|c| max|ratio| and
 *                  meets 1e-5 sum|c| only where the terms of a row largely cancel — measured on the Jordan-Wigner
 *                  chemistry Hamiltonians of the five configured workloads: max 0.14 x the bound over 32 oracle rows and 0.31 x
 *                  over 1,101 rows against the fp32 path at 76 qubits, 0.42 x / 0.66 x at 52 qubits.  On other
 *                  Hamiltonians at hidden >= 384 it does NOT meet that bound (measured 1.5 x on a symmetry-sparse
 *                  20-qubit Hamiltonian with a one-hidden-layer net, 2-3 x on generic Pauli lists): a caller who needs
 *                  1e-5 sum|c| there passes NQS_PATH_SIMT (fp32, ~30 x slower) and can check stats[4] = max|ratio|.
 *                  hidden (padded) <= 256 runs in SPLIT precision — every fp16 operand as hi + lo parts, three MMA
 *                  passes (hi.hi + lo.hi + hi.lo) — because a single fp16 pass misses the bound there (2 x); split
 *                  results are as accurate as the fp32 path (0.03 x the bound) at 3 x the tensor work.
 *  NQS_PATH_AUTO : TC when the shape supports it, else SIMT.  If the tensor-core weight pack of a supported shape cannot be
 *                  built or uploaded (device memory), the handle becomes an fp32-path handle: AUTO runs SIMT, a forced
 *                  NQS_PATH_TC returns NQS_EUNSUPPORTED, and nqs_made_path reports it from then on.
 * A handle (nqs_made_t / nqs_ham_t) owns device scratch that its compute calls reuse: use one handle from one
 * host thread and one CUDA stream at a time, on the device that was current when it was first used (other
 * devices: NQS_EINVAL). */
enum nqs_path { NQS_PATH_AUTO = 0, NQS_PATH_SIMT = 1, NQS_PATH_TC = 2 };

/* ---- (a1) Hamiltonian compile: Fig. 1 (:101) -------------------------------------
 * "we constructed a string parser that computes an Operator Matrix along with coefficients ... collect
 * the indices of sigma_1, sigma_2 operators prior to the training and only keep a buffer of unique
 * flippings and their corresponding number of occurrences".
 *
 * codes  : host uint8 [n_terms][n_qubits], the Operator Matrix, entries 0..3.
 * coeffs : host double [n_terms], real alpha_p (:47).
 * Result (host copy kept for nqs_ham_export; device copy made on first compute call):
 *   1. per term (f, s) and r = popcount(f & s);
 *   2. terms with identical (f, s) merged, coefficients summed in fp64 in input order, left to right;
 *   3. nothing dropped except a merged coefficient that is exactly 0.0;
 *   4. groups = distinct f, ascending as unsigned 128-bit integers (word 1 major); inside a group terms
 *      ascending by s the same way; offsets[g] .. offsets[g+1] index the terms of group g;
 *   5. coef = (float)c round-to-nearest-even; ycount = r.
 * n_terms = 0 is valid (E_loc = 0).  Pure host work: usable without a GPU. */
int nqs_ham_compile(int n_qubits, int64_t n_terms, const uint8_t *codes, const double *coeffs,
                    nqs_ham_t **out);

/* Same, from bit-packed incidence rows: fmask = F^{1,2}, smask = F^{2,3}, host uint64 [n_terms][2]. */
int nqs_ham_compile_packed(int n_qubits, int64_t n_terms, const uint64_t *fmask, const uint64_t *smask,
                           const double *coeffs, nqs_ham_t **out);

/* Same, from text (the paper's Hamiltonians are "stored in a string format", parsed by a "string
 * parser", :154; the syntax is not given -- reading A4): one term per line, the real coefficient first (plain,
 * parenthesised, or a complex literal with zero imaginary part such as "(0.5+0j)"), then either a dense word of
 * n_qubits letters from IXYZ (letter j = qubit j) or sparse factors "X0 Y3 Z12"; '[' ']' '*' ',' separate, '#'
 * comments.  The coefficient is a plain decimal literal ("-0.25", "1.5e-3") read independently of the locale; hex
 * literals, "nan", "inf" and literals that overflow a double are refused.  Malformed lines, a qubit named twice (an
 * explicit I counts as naming it) or a non-zero imaginary part: NQS_EINVAL. */
int nqs_ham_compile_text(int n_qubits, const char *text, nqs_ham_t **out);

/* K = merged term count, G = number of unique flips, sum_abs_coeff = sum_t |c_t| (fp64, merged, the
 * tolerance scale of BASELINE.json).  Any output pointer may be NULL. */
int nqs_ham_info(const nqs_ham_t *ham, int *n_qubits, int64_t *K, int64_t *G, double *sum_abs_coeff);

/* Host copies of the grouped tensors (for bit-exact tests).  Caller-allocated:
 * flips uint64 [G][2], offsets uint32 [G+1], zy uint64 [K][2], ycount uint8 [K], coef float [K].
 * Any pointer may be NULL. */
int nqs_ham_export(const nqs_ham_t *ham, uint64_t *flips, uint32_t *offsets, uint64_t *zy,
                   uint8_t *ycount, float *coef);

void nqs_ham_free(nqs_ham_t *ham);

/* ---- model parameters: PAPER.md:84 (architecture), :86 (masks "remove the connections"), :107 ------
 * n_hidden_layers : 1 (the paper's diagram) or 2 (BASELINE.json configs).
 * order      : host int32 [n] permutation; autoregressive position d reads qubit order[d]
 *              (NULL = identity; the paper's default is reverse, :107).
 * deg_hidden : host int32 [n_hidden_layers][hidden], MADE degrees in [1, n-1]
 *              (NULL = 1 + floor(j*(n-1)/hidden) for every layer).
 *              Masks: M1[j][d] = deg1[j] >= d+1;  Mk[j'][j] = deg_k[j'] >= deg_{k-1}[j];
 *              Mout[d][j] = d+1 > deg_L[j].
 * weights    : n_hidden_layers+1 host fp32 matrices, row-major [out][in], UNMASKED:
 *              [hidden][n], ([hidden][hidden]), [n][hidden]; columns/rows indexed by position d.
 * biases     : matching host fp32 vectors.
 * phase_weights / phase_biases : [hidden][n-2], [4][hidden] / [hidden], [4]; the phase net reads
 *              u_d = 2 z_d - 1 for positions d < n-2 and phi = o[2 z_{n-2} + z_{n-1}].
 * Pure host work (masking, packing, fp16 splitting); device copies are made on first compute call. */
int nqs_made_create(int n_qubits, int hidden, int n_hidden_layers, const int32_t *order,
                    const int32_t *deg_hidden, const float *const *weights, const float *const *biases,
                    const float *const *phase_weights, const float *const *phase_biases,
                    nqs_made_t **out);

/* Hamming-weight constraint of the model: PAPER.md:109-120 (Eq. 11-13), :136-142 (Eq. 14).  With n_up, n_down >= 0 the
 * wavefunction is the CONSTRAINED one: every conditional that Eq. 14 clamps to 0 or 1 (reading A13, see
 * nqs_made_sample) contributes log 1 = 0 to log|psi| = 1/2 sum_d log pi_hat_d, and a configuration that violates Eq. 12
 * (even qubits = up spins, odd = down) has psi = 0: nqs_made_logpsi returns log|psi| = -inf for it and it contributes
 * ratio 0 to nqs_local_energy.  nqs_energy_grad differentiates the same function (clamped logits get no gradient).
 * n_up = n_down = -1 (the state after nqs_made_create) switches the constraint off: raw sigmoid conditionals (A12). */
int nqs_made_set_constraint(nqs_made_t *made, int n_up, int n_down);

/* Host copy of the masked fp32 weight W_k (.) M_k of layer k (0-based, k <= n_hidden_layers), row-major
 * [out][in] in position order — lets a CPU test check the mask rule without a GPU. */
int nqs_made_export_masked(const nqs_made_t *made, int layer, float *out);

void nqs_made_free(nqs_made_t *made);

/* Which kernels `path` resolves to for this model: NQS_PATH_SIMT or NQS_PATH_TC, or a negative status
 * (NQS_EUNSUPPORTED when NQS_PATH_TC is forced on an unsupported shape).  Host only. */
int nqs_made_path(const nqs_made_t *made, int path);

/* Bookkeeping for the roofline report: multiply-add flops per psi evaluation that
 * NQS_PATH_TC ISSUES to the tensor cores (masked-zero K-steps skipped, padding and the bias K-steps included) and
 * the flops of the same chain with nothing skipped.  Needs a device (the weight images are packed on first use);
 * NQS_EUNSUPPORTED when the shape has no tensor-core path.  Host only, no kernel launch. */
int nqs_made_tc_flops(const nqs_made_t *made, int64_t *issued_per_eval, int64_t *dense_per_eval);

/* ---- (a4) MADE forward: Eq. 10 ---------------------------------------------------------
 * configs_dev : device uint64 [B][2]; bits >= n_qubits must be zero.
 * out_dev     : device float [B][2] = (log|psi|, phi); phi is not wrapped to [0, 2 pi).
 * Asynchronous on `cuda_stream`.  B = 0 is a no-op. */
int nqs_made_logpsi(const nqs_made_t *made, const uint64_t *configs_dev, int64_t B, float *out_dev,
                    int path, void *cuda_stream);

/* ---- (a3) Pauli contraction alone: Eq. 16 summed inside each unique-flip group --------
 * S[i][g - g0] = sum_{t in group g} c_t (-i)^{r_t} (-1)^{popcount(x_i & s_t)},  g in [g0, g1).
 * samples_dev : device uint64 [B][2];  S_out_dev : device float [g1-g0][B][2] (Re, Im), group-major: the B sums of
 * one group are contiguous.
 * Provided for tests and for the contraction-only throughput figure; nqs_local_energy fuses this step
 * and never materialises S. */
int nqs_pauli_contract(const nqs_ham_t *ham, const uint64_t *samples_dev, int64_t B, int64_t g0,
                       int64_t g1, float *S_out_dev, void *cuda_stream);

/* ---- (a2-a7) local energy: PAPER.md:122-134 Alg. 1, :152 Eq. 15, :200 Eq. 17, :202 mini-batches ----
 * samples_dev  : device uint64 [B][2] (unique samples; duplicates are harmless).
 * counts_dev   : device int64 [B] multiplicities (:105 "counter"), or NULL = all ones.  They weight the
 *                statistics only; E_loc does not depend on them.
 * minibatch    : samples per pass (gradient-accumulation slice, :202); 0 = auto (8192).  A pure partition
 *                in row order, last slice may be short.
 * eloc_out_dev : device float [B][2] = (Re, Im) of l_theta(x_i).
 * stats_out_host : host double [5] = { sum n, sum n Re E, sum n Im E, sum n |E|^2, max |psi ratio| }
 *                or NULL.  When non-NULL the call synchronises the stream before returning; otherwise it
 *                is asynchronous.
 * Overflow of exp(delta log|psi|) propagates as inf/NaN into eloc; never an error code. */
int nqs_local_energy(const nqs_ham_t *ham, const nqs_made_t *made, const uint64_t *samples_dev,
                     const int64_t *counts_dev, int64_t B, int64_t minibatch, int path,
                     float *eloc_out_dev, double *stats_out_host, void *cuda_stream);

/* Same computation with HOST buffers: copies samples/counts host->device, runs nqs_local_energy on an
 * internal stream, copies eloc device->host and synchronises.  samples_host uint64 [B][2], counts_host
 * int64 [B] or NULL, eloc_out_host float [B][2], stats_out_host double [5] or NULL.  A sample with a bit >= n_qubits set,
 * or a Hamiltonian and a model of different n_qubits: NQS_EINVAL (checked on the host before anything is launched; the
 * device-pointer entry points take "bits >= n_qubits are zero" as a precondition — checking it there would force a
 * synchronisation). */
int nqs_local_energy_host(const nqs_ham_t *ham, const nqs_made_t *made, const uint64_t *samples_host,
                          const int64_t *counts_host, int64_t B, int64_t minibatch, int path,
                          float *eloc_out_host, double *stats_out_host);

/* ---- (a6) statistics without any device allocation: PAPER.md:200 Eq. 17, :105 (counter) -------------------------
 * For callers that cannot let this library call cudaMalloc: a training loop whose framework allocator (PyTorch's
 * caching allocator, or an arena sized to the card) already owns all free device memory, so that a raw allocation
 * here fails or starves the framework later; a loop that overlaps several streams and cannot afford the device-wide
 * synchronisation cudaMalloc / cudaFree imply; a process held to a fixed device-memory budget (an MPS client with a
 * memory limit, ranks sharing a MIG slice).  Every other compute entry point grows a workspace inside the model
 * handle on first use; this one allocates nothing, ever — no cudaMalloc, cudaFree, events, streams or library calls
 * that allocate.
 *   eloc_dev      device float [B][2] = (Re, Im) of the local energies (the output of nqs_local_energy);
 *   counts_dev    device int64 [B] multiplicities, or NULL = all ones;
 *   stats_out_dev device double [4] = { sum n, sum n Re E, sum n Im E, sum n |E|^2 }, overwritten (the first four
 *                 entries of nqs_local_energy's stats; memory the caller owns, like the inputs);
 *   B             0 <= B <= NQS_STATS_STATIC_MAX_ROWS; more rows: NQS_ERANGE, nothing launched.  B = 0 writes zeros.
 * Asynchronous on `cuda_stream`; fp64, fixed summation order (bit-reproducible, unlike an atomic sum).
 * Scratch: per-CTA partial sums live in a 33 KB array that is part of the library's device image (one slot per 2048
 * rows, 1024 slots — that is where the row limit comes from).  Every GPU the process uses with libnqs loaded keeps
 * that array until exit.  Consequences for the caller:
 *   - the first call made with a given device current looks the array's device address up and caches it; make that
 *     first call during set-up, before any stream capture on that device;
 *   - all calls on one device share the array.  The library clears the one word that must start at zero on the
 *     call's stream, so back-to-back calls on ONE stream are fine; two calls that can overlap on the GPU (different
 *     streams without an ordering between them) race on it and both results are undefined.
 * Errors: NQS_EINVAL (NULL pointer, B < 0), NQS_ERANGE (B above the limit), NQS_EARCH / NQS_ECUDA (no sm_100 device,
 * a runtime call failed), NQS_EUNSUPPORTED (device ordinal >= 64). */
#define NQS_STATS_STATIC_MAX_ROWS 2097152   /* 2^21 = 1024 scratch slots x 2048 rows */
int nqs_weighted_stats_static(const float *eloc_dev, const int64_t *counts_dev, int64_t B,
                              double *stats_out_dev, void *cuda_stream);

/* ---- gradient of the energy objective: PAPER.md:71 Eq. 7, :73 (baseline), :202 (accumulation) ----------
 *   grad L(theta) = Re E[(l_theta(x) - b) conj(grad_theta log f(x))],   b = E[l_theta(x)],
 * the expectation taken over the unique samples weighted by their multiplicities (:105, :200).  log f = log|psi| + i phi
 * (:96 Eq. 10), so the MADE parameters receive Re(E - b) through log|psi|, the phase-net parameters Im(E - b) through phi.
 *
 * nqs_made_num_params : number of parameters = length of the flat gradient.  Flat order: for k = 0..n_hidden_layers:
 *   W_k (row-major [out][in]) then b_k; then P1 [hidden][n-2], c1 [hidden], P2 [4][hidden], c2 [4] -- the tensors of
 *   nqs_made_create in its argument order.  The gradient is with respect to the UNMASKED weights nqs_made_create takes:
 *   masked entries receive exactly 0.
 * nqs_energy_grad :
 *   samples_dev  device uint64 [B][2];  counts_dev device int64 [B] or NULL (= ones);
 *   eloc_dev     device float [B][2], the local energies of these samples (the output of nqs_local_energy);
 *   minibatch    rows per accumulation pass (0 = 8192): bounds the workspace (~ 6 * hidden * minibatch floats);
 *   global_stats_host  NULL, or host double [3] = { sum n, sum n Re E, sum n Im E } over the samples of ALL
 *                data-parallel replicas (:146): b and the normalisation are then taken from it, so that the SUM of the
 *                replicas' gradients is the gradient of the whole batch (paper_2208_05637_b200/distributed.py);
 *   grad_out_dev device float [n_params], overwritten;
 *   baseline_out_host host double [2] = (Re b, Im b) or NULL; when non-NULL the call synchronises the stream.
 * fp32 on CUDA cores (the B sampled rows are ~1e-5 of the E_loc work), fixed reduction order: bit-reproducible.
 * B = 0 gives a zero gradient.
 * Preconditions the call cannot check without synchronising: the total count sum n is positive (0 gives NaN), and —
 * when the handle carries a constraint — every sample satisfies Eq. 12 (the sampler produces only such rows; a
 * violating row has psi = 0, its gradient is undefined and the value written for it is unspecified).
 * global_stats_host[0] must be the true total over all replicas; <= 0 is NQS_EINVAL.  One row tile needs
 * (2 npad + 3 hidden + 6) * 64 B of shared memory; that fits 227 KB for every shape nqs_made_create accepts
 * (hidden <= 1024, n <= 128: 213 KB), and a shape that did not would get NQS_EUNSUPPORTED before anything is launched. */
int nqs_made_num_params(const nqs_made_t *made, int64_t *n_params);
int nqs_energy_grad(const nqs_made_t *made, const uint64_t *samples_dev, const int64_t *counts_dev,
                    const float *eloc_dev, int64_t B, int64_t minibatch, const double *global_stats_host,
                    float *grad_out_dev, double *baseline_out_host, void *cuda_stream);

/* ---- batched autoregressive sampler: PAPER.md:105-107, :109-120, :136-142 (Eq. 11-14) -----------------------
 * "keep track of a sample buffer ... associated with a counter storing the number of occurrences ... At each of the
 * n iterations, we first double the size of the buffer ... update the counter ... through Bernoulli sampling with
 * probabilities computed by forward pass ... eliminate the samples ... that have the lowest numbers of occurrences."
 * Positions are visited in the model's autoregressive order (the paper's reversed order, :107, is `order` of
 * nqs_made_create).  Readings where the paper is silent or garbled (A13 / A25):
 *   - the split of a counter of c occurrences is c Bernoulli trials, one per DRAW s in [0, n_draws): at position d the
 *     draw uses u = (w + 1/2) 2^-32, w = first word of Philox4x32-10(key = (seed lo, seed hi), counter = (s lo, s hi,
 *     d, 0)), and takes bit 1 iff u < pi_hat (conditionals in fp32) -- replayable, independent of buffer order;
 *   - children of buffer entry i sit at 2i (bit 0) and 2i + 1 (bit 1); zero counters leave the buffer; if more than
 *     max_unique remain the largest counters stay (ties: buffer order) and the other draws are discarded
 *     (max_unique = 0: no elimination);
 *   - n_up, n_down >= 0 switch on the Hamming-weight clamp of Eq. 14 (even qubits = up spins, odd = down, Eq. 12): at
 *     a position of spin s with c spin-s bits already set and m spin-s positions left, pi_hat(1) = 0 if c = n_s,
 *     = 1 if n_s - c = m, else the network's conditional.  n_up = n_down = -1: the constraint of the handle
 *     (nqs_made_set_constraint), unconstrained if it has none.  A handle WITH a constraint only samples that
 *     constraint (a different pair: NQS_EINVAL), so samples, log psi, E_loc and gradient share one pi_hat; on a handle
 *     without one the pair clamps the sampler alone.
 * samples_out_dev : device uint64 [cap][2], counts_out_dev : device int64 [cap], cap = max_unique if 0 < max_unique <
 *   n_draws else n_draws; the first *n_unique_out_host rows are written, in buffer order (unique, bit j = qubit j).
 * Synchronous (n readbacks of the buffer size); its buffers live in the model handle and grow on demand (a handle
 * serves one nqs_made_sample call at a time).  n_draws < 2^30
 * (buffer indices are 32-bit; more: NQS_ERANGE). */
int nqs_made_sample(const nqs_made_t *made, int64_t n_draws, uint64_t seed, int n_up, int n_down,
                    int64_t max_unique, uint64_t *samples_out_dev, int64_t *counts_out_dev,
                    int64_t *n_unique_out_host, void *cuda_stream);

/* Number of kernels this library has launched in the calling process since load (monotonic). */
int64_t nqs_kernel_launch_count(void);

/* Duration in milliseconds of the dominant (MADE-chain) kernel launches of the LAST nqs_local_energy /
 * nqs_local_energy_host call, summed over its mini-batches, measured with CUDA events on the launching
 * stream; *n_launches receives how many launches that was.  Synchronises on those events. */
int nqs_last_chain_kernel_ms(const nqs_made_t *made, float *ms, int *n_launches);

const char *nqs_strerror(int status);

#ifdef __cplusplus
}
#endif
#endif /* NQS_H_ */
