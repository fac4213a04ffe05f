/*
 * nep.h -- C ABI of libnep_b200: one training step of a neuroevolution potential (NEP) on one B200.
 *
 * The calls follow the paper's statement of the problem (arxiv/paper_2606_19557, "TorchNEP").
 * P:NNN = line NNN of the paper text; "DESIGN C<k>" = DESIGN.md section 3, step k.
 *
 *   model inputs   : species, cutoffs, n_max, basis sizes, l_max, neurons        Table I
 *   data           : positions, boxes, types, energy / force / virial labels      Eqs. 5-7
 *   geometry cache : neighbour lists, displacement vectors, basis aggregates,
 *                    built once and kept on the GPU
 *   step           : descriptors (Eqs. 15-20) -> network (Eq. 3) -> E, F, W ->
 *                    loss (Eqs. 4-7) -> analytic gradient (Eq. 8) -> Adam  Eqs. 9-13
 *
 * Conventions
 *   - Opaque context; one context = one CUDA device + one stream; not thread-safe per context.
 *   - Every call returns 0 (NEP_OK) or a negative NEP_E* code; nep_last_error() gives the message
 *     (NUL-terminated, owned by the context, valid until the next call on it).  No C++ exception
 *     crosses the ABI.  Nothing is truncated silently: exceeding a capacity is NEP_ECAPACITY.
 *   - "host" pointers are plain host memory, borrowed for the duration of the call only.
 *     "device" pointers are CUDA device memory on the context's device.
 *   - Device memory is obtained through the caller's allocator callbacks (the Python binding
 *     implements them with torch tensors).  The library never calls cudaMalloc: alloc == NULL or
 *     free_ == NULL is NEP_EINVAL.
 *   - Step calls (nep_forward / nep_loss_grad / nep_adam_step) enqueue work on the context's stream
 *     and return without synchronising unless a host output is requested.
 *   - There is no CPU fallback: without a CUDA device nep_create fails with NEP_ECUDA.
 *
 * Layouts (DESIGN C0)
 *   theta  : for each species t: w0[t] (neurons x D, row-major), b0[t] (neurons), w1[t] (neurons);
 *            then b1; then cR[t_i][t_j][n][k]; then cA[t_i][t_j][n][k].   n = 0..n_max, k = 0..basis_size.
 *   q      : radial n -> n; 3-body (l, n) -> n_R + (l-1) n_A + n; 4-body n -> n_R + l3 n_A + n; 5-body next.
 *   box    : 9 doubles per structure, rows are the cell vectors a, b, c.
 *   virial : 9 values per structure, row-major xx xy xz yx yy yz zx zy zz; W = -sum d (x) dE/dd (eV).
 */
#ifndef NEP_B200_H
#define NEP_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NEP_OK 0
#define NEP_EINVAL (-1)    /* bad argument */
#define NEP_ESTATE (-2)    /* call out of order */
#define NEP_ECUDA (-3)     /* CUDA runtime error (message holds cudaGetErrorString) */
#define NEP_ENOMEM (-4)    /* allocator returned NULL */
#define NEP_ECAPACITY (-5) /* an internal capacity would be exceeded */

typedef struct nep_ctx nep_ctx;

/* Device allocator callbacks.  alloc returns a device pointer aligned to >= 256 bytes, or NULL. */
typedef void* (*nep_alloc_fn)(void* user, size_t nbytes);
typedef void (*nep_free_fn)(void* user, void* ptr);

/* Library version string, e.g. "nep_b200 0.1 (sm_100a)". */
const char* nep_version(void);

/* Model definition (Table I).  1 <= n_species <= 16 (the paper's largest set);
 * 0 < rc_A <= rc_R (DESIGN G22); n_max >= 0; 1 <= basis <= 16; l_max_3b in 1..4 (three-body orders l = 1..l_max_3b;
 * Table I uses 4); l_max_4b in {0,2}; l_max_5b in {0,1} (Table I: "l_max 4 2 1"); neurons >= 1.
 * cuda_stream: a cudaStream_t (NULL = default stream).  alloc/free_/alloc_user: see above.
 * On success *out owns the context; release with nep_destroy. */
int nep_create(nep_ctx** out, int n_species, double rc_R, double rc_A, int n_max_R, int n_max_A,
               int basis_R, int basis_A, int l_max_3b, int l_max_4b, int l_max_5b, int neurons,
               nep_alloc_fn alloc, nep_free_fn free_, void* alloc_user, void* cuda_stream);

/* A model as a file, and prediction with it ("prediction").  nep_save_model writes the hyper-parameters of
 * Table I, the scaler of Eq. 2 [D] and theta [N_par, layout of DESIGN C0] as text:
 *     nep_b200_model 1 / n_species T / cutoff rc_R rc_A / n_max R A / basis_size R A / l_max l3 l4 l5 / neuron H /
 *     scaler D, D values / theta N_par, N_par values (9 significant digits: fp32 values round-trip exactly).
 * The keywords are those of the paper's input file (Table I); the layout is this library's own (the paper does not print the
 * layout of GPUMD's model files, DESIGN reading G28).  Needs parameters and a scaler (NEP_ESTATE otherwise).
 * nep_create_from_model_file = nep_create with the file's hyper-parameters + nep_set_params + nep_set_scaler; NEP_EINVAL if
 * the file cannot be read or is inconsistent.  Prediction is then nep_load_structures (labels NULL) + nep_build_neighbors +
 * nep_forward.  nep_get_model returns the hyper-parameters of a context (any pointer may be NULL): rc2 = {rc_R, rc_A},
 * n_max2, basis2 = {radial, angular}, l_max3 = {l_max_3b, l_max_4b, l_max_5b}. */
int nep_save_model(nep_ctx* ctx, const char* path);
int nep_create_from_model_file(nep_ctx** out, const char* path, nep_alloc_fn alloc, nep_free_fn free_, void* alloc_user,
                               void* cuda_stream);
int nep_get_model(const nep_ctx* ctx, int* n_species, double* rc2, int* n_max2, int* basis2, int* l_max3, int* neurons);

/* Releases every device buffer through free_ and the context itself.  NULL is a no-op. */
int nep_destroy(nep_ctx* ctx);

/* Message of the last failing call on ctx ("" if none).  ctx == NULL: message of a failed nep_create. */
const char* nep_last_error(const nep_ctx* ctx);

/* D = (n_max_R+1) + (n_max_A+1) * (l3 + [l4>0] + [l5>0])  and
 * N_par = T (D+2) H + 1 + T^2 [(n_max_R+1)(basis_R+1) + (n_max_A+1)(basis_A+1)]   (pinned by Table II). */
int nep_num_descriptors(const nep_ctx* ctx);
int64_t nep_num_params(const nep_ctx* ctx);

/* Structures and labels (host, copied to the device).  Replaces any previously loaded set.
 *   n_atoms [S]; pos [sum N][3] Cartesian, Angstrom; box [S][9]; type [sum N] in 0..T-1;
 *   E [S] eV (total energy, Eq. 5); F [sum N][3] eV/A (Eq. 6); W [S][9] eV (Eq. 7);
 *   has_virial [S] 0/1 or NULL = all (DESIGN G14).  E, F, W may all be NULL (predict only; labels can be
 *   attached later with nep_set_labels).
 * NEP_EINVAL for non-finite input, det(box) <= 0, type out of range, or a position whose fractional
 * coordinate is outside [0,1) (wrap first; tolerance 1e-9). */
int nep_load_structures(nep_ctx* ctx, int n_struct, const int* n_atoms, const double* pos, const double* box,
                        const int* type, const double* E, const double* F, const double* W,
                        const unsigned char* has_virial);

/* Attach / replace labels of the loaded set (same shapes as above; all three required). */
int nep_set_labels(nep_ctx* ctx, const double* E, const double* F, const double* W, const unsigned char* has_virial);

/* S0a + S0b: neighbour lists of every loaded structure for both cutoffs -- all periodic
 * images (j, n) != (i, 0) with |d| < rc, d = (((r_j - r_i) + n_a a) + n_b b) + n_c c in IEEE fp64 without
 * FMA (DESIGN C1), ascending (j, n_a, n_b, n_c) per atom -- then the per-pair geometry cache and the
 * per-atom radial basis aggregate.  Selects the full set as the current batch. */
int nep_build_neighbors(nep_ctx* ctx);

/* Reads the lists back to the host (parity checks need no internals).  which: 0 = radial, 1 = angular.
 * Two-call pattern: with j == NULL only *n_pairs and offsets (if non-NULL) are written.
 * offsets [sum N + 1] (int64); j [P] = neighbour index local to the structure; shift [P][3] = (n_a,n_b,n_c). */
int nep_get_neighbors(nep_ctx* ctx, int which, int64_t* n_pairs, int64_t* offsets, int* j, signed char* shift);

/* Parameters, gradient and optimiser state: host arrays of N_par floats, layout above.
 * nep_get_grad returns g = grad_theta L of the last nep_loss_grad (Eq. 8). */
int nep_set_params(nep_ctx* ctx, const float* theta);
int nep_get_params(nep_ctx* ctx, float* theta);
int nep_get_grad(nep_ctx* ctx, float* g);
/* Overwrites the stored gradient (parity runs feed the same g to both optimisers; also allows external gradients). */
int nep_set_grad(nep_ctx* ctx, const float* g);
int nep_set_adam_state(nep_ctx* ctx, const float* m, const float* v, const float* vmax, int64_t t);
int nep_get_adam_state(nep_ctx* ctx, float* m, float* v, float* vmax, int64_t* t);

/* Descriptor scaler of Eq. 2: s = 1 / (max - min) of each component over every atom of the
 * loaded set at the current parameters; constant afterwards (no gradient flows through it).
 * compute needs neighbours and parameters; set/get exchange D doubles with the host. */
int nep_compute_scaler(nep_ctx* ctx);
int nep_set_scaler(nep_ctx* ctx, const double* s);
int nep_get_scaler(nep_ctx* ctx, double* s);
/* Eq. 2 when the training set is spread over several contexts (data-parallel training, below): the range of Eq. 2 is
 * over EVERY atom of the set, so each context reports the minimum and maximum of each descriptor component over its
 * own atoms (qmin, qmax: D doubles each, host; +inf / -inf for a context without atoms), the caller reduces them
 * over the contexts (element-wise min / max, e.g. two all-reduces) and hands the result to every context, which
 * forms s = 1 / (max - min) itself (a component without a range gets s = 1, DESIGN G10).
 * nep_compute_scaler == nep_compute_descriptor_range followed by nep_set_scaler_from_range on one context.
 * Both select the full loaded set as the current batch. */
int nep_compute_descriptor_range(nep_ctx* ctx, double* qmin, double* qmax);
int nep_set_scaler_from_range(nep_ctx* ctx, const double* qmin, const double* qmax);

/* Eq. 2 without a context and without an allocator: s_v = 1 / (max_i q_v^i - min_i q_v^i) for v = 0..n_desc-1 over
 * the n_atoms rows of a descriptor matrix that already sits on the device.  Who needs it: every other call here takes its device
 * memory from the nep_alloc_fn a context was created with, so a caller that has no allocator to lend -- its framework's pool owns
 * the whole GPU and a raw cudaMalloc would fail, it is in the middle of stream-ordered work that cudaMalloc's device-wide
 * synchronisation would stall, or it is plain C / Fortran holding two device pointers and nothing else -- cannot use
 * nep_compute_scaler.  This call allocates nothing, on the device or through any library: its working memory is an array of
 * NEP_STATIC_SCRATCH_BYTES that is part of the library image (each GPU that loads the library keeps it until the process ends).
 *   q_dev  [n_atoms][n_desc] float, device, row-major, unscaled descriptors (the layout nep_get_descriptors returns);
 *   s_dev  [n_desc] float, device, written by the kernel; a component without a range (all rows equal, or n_atoms == 0) gets 1,
 *          by the same fp32 rule as nep_compute_scaler (DESIGN G10);
 *   cuda_stream: a cudaStream_t (NULL = default stream) on the CURRENT device, which must also own q_dev and s_dev; the work is
 *          enqueued there and the call returns without synchronising.  Both buffers stay the caller's.
 * Limits and sharing: n_desc <= NEP_STATIC_MAX_DESCRIPTORS (NEP_ECAPACITY beyond, nothing launched); n_atoms is not limited.
 * All calls on a device use the one array: calls whose kernels could run at the same time on that GPU (two streams, two
 * threads) race and must be serialised by the caller; calls in stream order are fine, nothing has to be cleared in between.
 * The first call on each device looks up the array's address and caches it: make it before, not during, a stream capture.
 * Errors: NEP_EINVAL (n_desc < 1, n_atoms < 0, NULL pointer), NEP_ECAPACITY, NEP_ECUDA; the message is nep_last_error(NULL)
 * (per host thread, shared with nep_create's). */
#define NEP_STATIC_MAX_DESCRIPTORS 128
#define NEP_STATIC_SCRATCH_BYTES 303360
int nep_scaler_static(const float* q_dev, int64_t n_atoms, int n_desc, float* s_dev, void* cuda_stream);

/* Mini-batch = a list of structure ids ("batch" of Table I).  ids == NULL: the whole set.
 * ids are copied to the device; the same id must not appear twice.  Selecting the batch that is already current (full-batch
 * training does so every step) uploads its tables again but keeps the tables derived from them on the device. */
int nep_set_batch(nep_ctx* ctx, int n, const int* struct_ids);

/* S1-S5: descriptors, network, energies (Eq. 1), forces and virials (P:145 closed forms) of the batch.
 *   E_out [S_b], F_out [N_b][3], W_out [S_b][9], all float, in batch order (atoms in the order of ids);
 *   each may be NULL.  outputs_on_host != 0: host pointers (the call synchronises); else device pointers.
 * Results are kept inside the context for nep_loss_grad. */
int nep_forward(nep_ctx* ctx, void* E_out, void* F_out, void* W_out, int outputs_on_host);

/* Short-range pair correction ("TorchNEP fully supports the Ziegler-Biersack-Littmark (ZBL) potential [24] as a short-range
 * correction").  The paper prints neither the screening constants nor the switching radii, so the library stores
 * none: the term has a fixed form, a screened Coulomb repulsion that is switched off smoothly, and the caller supplies every
 * number in it (DESIGN reading G29):
 *     E += sum over undirected pairs {(i,0), (j,n)} with r < r_outer of  phi_ij(r),
 *     phi_ij(r) = sw(r) (coulomb_k Z_i Z_j / r) sum_{m < n_terms} coef[m] exp(-expo[m] r / a_ij),  a_ij = a_prefac / (Z_i^a_pow + Z_j^a_pow),
 *     sw(r) = 1 for r <= r_inner, 1/2 (1 + cos(pi (r - r_inner) / (r_outer - r_inner))) up to r_outer, 0 beyond.
 * Z [n_species] > 0 (host); 0 <= r_inner < r_outer <= rc_R (Angstrom); 1 <= n_terms <= 8, expo >= 0 (host arrays, copied);
 * a_prefac > 0 (Angstrom); coulomb_k = e^2 / (4 pi eps_0) in eV Angstrom.  From then on nep_forward adds the term to E, F and W
 * (F = -dE/dr, W = -sum d (x) dE/dd); nep_loss_grad sees the corrected predictions; the term holds no model parameter, so it adds
 * nothing to the gradient by itself.  Z == NULL or n_terms == 0 switches it off.  Not written to model files.  Invalidates the
 * step graph and the forward results.  NEP_EINVAL / NEP_ECAPACITY for arguments outside the ranges above. */
int nep_set_pair_correction(nep_ctx* ctx, const double* Z, double r_inner, double r_outer, int n_terms, const double* coef,
                            const double* expo, double a_prefac, double a_pow, double coulomb_k);

/* Unscaled descriptors q [N_b][D] (float, host) of the current batch, from the last nep_forward. */
int nep_get_descriptors(nep_ctx* ctx, float* q);

/* S6-S9: L = lE dE + lF dF + lV dV (Eqs. 4-7, batch normalisers) and g = grad_theta L with respect to every
 * network weight and descriptor coefficient (Eq. 8; DESIGN C9-C12).  Needs nep_forward on the same batch
 * and parameters immediately before (NEP_ESTATE otherwise) and labels.  loss4_host: {L, dE, dF, dV} as
 * doubles on the host (synchronises) or NULL (stays on the device; see nep_get_loss). */
int nep_loss_grad(nep_ctx* ctx, double lambda_E, double lambda_F, double lambda_V, double* loss4_host);
int nep_get_loss(nep_ctx* ctx, double* loss4_host);   /* valid until the next nep_forward, also after nep_adam_step */

/* Data-parallel training over several contexts, one per GPU.  Structures interact only with
 * themselves (Eq. 1), so the batch of a step is split by structure: every context holds its share of the data
 * set and calls nep_set_batch with its share of the batch.  The loss of Eq. 4 and its gradient (Eq. 8) are sums over
 * structures and atoms divided by the batch counts of Eqs. 5-7, so with the counts of the WHOLE batch given here
 * (S_b structures, N_b atoms, S_v structures with virial labels; each >= this context's own count, NEP_EINVAL otherwise)
 * every context produces its additive share of {L, dE, dF, dV} and of g.  The caller sums g [N_par floats] and the four
 * loss terms [4 doubles] over the contexts in place -- device pointers from nep_grad_device_ptr, e.g. one NCCL
 * all-reduce each -- and then calls nep_adam_step on every context (identical updates, no parameter broadcast).
 * nep_set_batch and nep_set_labels reset the counts to those of the local batch.  Call after them, before nep_loss_grad. */
int nep_set_batch_normalisers(nep_ctx* ctx, int64_t n_struct_whole, int64_t n_atoms_whole, int64_t n_virial_whole);
int nep_grad_device_ptr(nep_ctx* ctx, float** g, double** loss4);

/* S10: Adam with AMSGrad on theta with the stored gradient.  variant 0 = Eqs. 9-13 literally (running max of
 * the bias-corrected second moment, epsilon inside the root); variant 1 = torch.optim.Adam(amsgrad=True).
 * Increments the step count t.  Invalidates the forward results. */
int nep_adam_step(nep_ctx* ctx, double lr, double beta1, double beta2, double eps, int variant);

/* One training step = nep_forward + nep_loss_grad + nep_adam_step on the current batch, without outputs (the loss terms stay
 * on the device: nep_get_loss).  use_graph != 0: the step's kernels are captured once into a CUDA graph and replayed with one
 * launch; loss weights, learning rate and the bias corrections of Eq. 11 are written into the graph's nodes before each
 * replay, so they may change from step to step.  nep_set_batch, nep_set_batch_normalisers, nep_set_labels,
 * nep_load_structures and nep_build_neighbors invalidate the graph (nep_set_batch only if the batch's shape or its number of atoms
 * per species changes); the first step after that runs as
 * the three calls, the graph is captured when the same batch is stepped a second time.  Same results as the three calls. */
int nep_train_step(nep_ctx* ctx, double lambda_E, double lambda_F, double lambda_V, double lr, double beta1, double beta2,
                   double eps, int variant, int use_graph);

/* Blocks until the context's stream is idle. */
int nep_synchronize(nep_ctx* ctx);

/* Measurement aids.  launch_count: kernels launched by this context since creation.
 * Profiling: when enabled, every kernel launch of the step calls is bracketed by CUDA events on the
 * context's stream; nep_profile_read returns, for up to `cap` distinct kernels, name pointers (static
 * strings), accumulated milliseconds and launch counts, and resets the accumulators.  Returns the number
 * of kernels through *n. */
int nep_launch_count(nep_ctx* ctx, int64_t* n);
int nep_profile_enable(nep_ctx* ctx, int on);
/* While paused no events are recorded (no synchronisation, accumulators kept): lets a caller time kernels on a sample
 * of its steps only, so that the event records do not sit between the kernels of every step. */
int nep_profile_pause(nep_ctx* ctx, int paused);
int nep_profile_read(nep_ctx* ctx, int cap, const char** names, double* ms, int64_t* launches, int* n);

/* 1 if the network kernels of this context (S3, S8) run as tcgen05 tiles, 0 if the model's tiles do not fit in shared memory /
 * tensor memory (or NEP_ANN_FFMA=1 was set when the context was created) and the FFMA tiles are used.  Tests use it to make sure a
 * parity case really exercises the tensor-core path. */
int nep_network_on_tensor_cores(const nep_ctx* ctx);

/* Measurement aid, no context: runs a register-resident FP32 FMA loop (32 independent chains per thread, 2048 threads per SM)
 * on the current device for a few milliseconds and returns the rate it reached in TFLOP/s (2 flops per FMA) -- the measured
 * counterpart of the derived FP32 peak bench.py's "alu" roofline divides by.  Synchronises cuda_stream. */
int nep_measure_fp32_peak(void* cuda_stream, double* tflops);

/* Sizes of the loaded set / current batch: {S, N, P_R, P_A, S_b, N_b, P_R_b, P_A_b}. */
int nep_get_sizes(nep_ctx* ctx, int64_t* sizes8);

#ifdef __cplusplus
}
#endif
#endif /* NEP_B200_H */
