/*
 * cos.h -- C-ABI of the B200-native CoS / SB-CoS DAG evaluator (arxiv 2507.12349, "CoS++").
 *
 * The library evaluates, for many Monte-Carlo configurations at once and in fp64, the connected
 * Hubbard Feynman-diagram sum S_n of PAPER.md Eq. 63 (SB-CoS, Algorithm 3) or
 * its flavour-uniform specialisation (Eq. 8-12), optionally for all 2^n-1
 * vertex subsets (terminal readouts, Eq. 13-15), by walking a compiled layered DAG
 * (Eq. 16).
 *
 * Conventions
 *   n        perturbative order = interaction vertices (1..COS_MAX_N); endpoints 2n (Eq. 58).
 *   N_f      number of flavours.
 *   n_sub    sublattices per vertex: 1 (square) or 2 (honeycomb, sublattice-SUMMED, Eq. 4, 55).
 *   d        n * n_sub; endpoint index a = i*n_sub + s for vertex i (0-based) on sublattice s.
 *   block    one d x d propagator matrix; uniform mode has ONE block, SB mode N_f blocks.
 *   "host"/"device" below says where a pointer must live.  All device pointers must belong to
 *   the CUDA device that was current when cos_build / cos_tab_build was called.
 *
 * Errors: every function returns a status (COS_OK = 0); nothing throws or aborts across the ABI.
 * cos_last_error() returns a thread-local human-readable message for the last failure.
 * There is NO CPU fallback: without a CUDA device cos_build succeeds only in host-only mode
 * (COS_BUILD_HOST_ONLY, used to inspect the compiled DAG) and cos_eval fails with COS_ECUDA.
 */
#ifndef COS_B200_H
#define COS_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define COS_MAX_N 12
#define COS_MAX_COLOURS 4          /* SB mode: N_f <= 4 (colour carried in the state) */

typedef struct cos_handle_s* cos_handle;     /* opaque: host DAG + device program + device workspace */
typedef struct cos_tab_s*    cos_tab;        /* opaque: device propagator lookup table */
typedef void*                cos_stream;     /* a cudaStream_t (0 / NULL = legacy default stream) */

enum { COS_OK = 0, COS_EINVAL = 1, COS_ENOMEM = 2, COS_ECUDA = 3, COS_EUNSUPPORTED = 4 };
enum { COS_LATTICE_SQUARE = 0, COS_LATTICE_HONEYCOMB = 1 };

/* flags for cos_build_ex / cos_build_orders (bitwise or) */
enum {
    COS_BUILD_HOST_ONLY = 1,       /* compile the DAG, do not touch CUDA (cos_eval then fails) */
    COS_BUILD_NO_FUSED = 2,        /* small DAGs: use the per-layer kernels instead of the single fused launch */
    COS_BUILD_UNIFORM_SHIFT = 4    /* uniform CoS WITH a counterterm: shifts[0] = sigma = alpha/U (see cos_build) */
};

/* ---- (1) DAG compiler: PAPER.md:160-265 (canonical keys Eq. 17, 79-80; pruning Eq. 19-24) ----------
 * Enumerates the reachable states (occupancy mask m_i in {0,(1,s),2}, head, endpoint, colour), prunes
 * them against the requested readouts, layers them by total occupancy and uploads the per-layer
 * program.
 *   n, n_flavors    as above.
 *   lattice         COS_LATTICE_SQUARE (n_sub=1) or COS_LATTICE_HONEYCOMB (n_sub=2).
 *   shifts          host, may be NULL.
 *                   NULL      -> uniform CoS: one propagator block, factor N_f per closed loop
 *                                (Eq. 12, 15), no counterterm.
 *                   non-NULL  -> SB-CoS: n_flavors blocks, shifts[lam] = sigma_lam = alpha_lam/U
 *                                (shift-close weight), n_flavors values; colour sums
 *                                replace N_f.  n_flavors <= COS_MAX_COLOURS.
 *                   With COS_BUILD_UNIFORM_SHIFT (cos_build_ex): uniform CoS with a counterterm (PAPER.md:431,
 *                   Eq. 33; reading G12 of DESIGN.md): one propagator block, factor N_f per closed loop, and
 *                   the true one-cycle v -> v weighs A[v][v] + sigma/N_f with sigma = shifts[0] (one value).
 *   readout_envelope 0 -> one output per configuration, the full-order value C_{[n]};
 *                   n -> all 2^n-1 subset values (Eq. 5 with N = n); anything else: COS_EINVAL.
 *   out             receives the handle; the caller releases it with cos_free.
 * The values returned by cos_eval follow the physical convention of Eq. 83 (no shift-shift term).
 * Structural limits (COS_EUNSUPPORTED, never COS_ENOMEM): n * n_sub <= 24; SB-CoS with more than COS_MAX_COLOURS
 * flavours; a propagator tile (n_blocks * d * d, + n_colours * d with shifts, entries of 256 bytes) that exceeds the
 * 226 KB of shared memory of one SM (e.g. honeycomb SB-CoS beyond n = 10 with two flavours); a layer of 2^24 - 1 or more
 * states (24-bit destination index of the layer program: honeycomb n >= 11).  COS_ENOMEM is host or device memory
 * exhaustion only.
 * What that covers: the square lattice at every order 1..12, uniform or SB with 2-4 flavours (tested on the GPU up to
 * n = 12 in both modes); honeycomb up to n = 10 in SB mode (two flavours: table 2*20*20 + 2*20 entries = 215 KB) and up
 * to n = 11 in uniform mode (92 M states, largest layer 15,990,424 < 2^24 - 1; tested on the GPU).  Beyond: SB honeycomb
 * n = 11 has a layer above 2^24 - 1 states AND a table of 2*22*22*256 B = 242 KB > 226 KB; uniform honeycomb n = 12 has a
 * layer above 2^24 - 1 states.  Both are limits of the layer program / kernel, not of device memory (a 16 M-state layer
 * needs 2 * 16 M * 256 B = 8.2 GB of slabs per batch tile, which fits many times).  */
int cos_build(int n, int n_flavors, int lattice, const double* shifts, int readout_envelope, cos_handle* out);
int cos_build_ex(int n, int n_flavors, int lattice, const double* shifts, int readout_envelope,
                 int flags, cos_handle* out);

/* Partial readout sets ("allowed orders U", Eq. 6; requested-output pruning Eq. 21-24):
 * all-subset layout (2^n-1 output rows, k = bitmask(S)-1), but only subsets whose order |S| has its bit set in
 * order_mask (bit k <-> |S| = k, 1 <= k <= n) are computed; states that reach no requested readout are pruned
 * (K_l = F_l ^ B_l, Eq. 23) and the rows of the other subsets are written as zeros by cos_eval.
 * order_mask without a bit in [1, n]: COS_EINVAL. */
int cos_build_orders(int n, int n_flavors, int lattice, const double* shifts, unsigned int order_mask, int flags,
                     cos_handle* out);

/* Compiler analysis (host only, no CUDA): future / past equivalence classes of the pruned DAG.
 * States with equal future signature Sigma+ (Eq. 25-26) could be merged by adding their values, states with equal past
 * signature Sigma- (Eq. 27-28) carry equal values and need to be stored once; operators are compared as SYMBOLS (the
 * propagator entry G_lambda[a][b] or the counterterm of colour lambda, with the integer coefficient of Eq. 17), i.e. for
 * generic numeric propagators.  One backward and one forward refinement pass.  Arguments as cos_build_ex (flags:
 * COS_BUILD_UNIFORM_SHIFT only).  out6 (host, 6 values): states, edges (E1..E4 uncoalesced + readouts), future classes,
 * edges after the future merge, past classes, edges after the past merge.  Limited to DAGs of at most 6e7 states
 * (COS_EUNSUPPORTED beyond).  DESIGN.md section 9 reports the result: the only equivalences of the reduced recurrence
 * are the N_c fresh-head states of a close-and-open step and the initial states -- both already exploited. */
int cos_equivalence_stats(int n, int n_flavors, int lattice, const double* shifts, int readout_envelope, int flags,
                          long long* out6);

/* ---- (3)+(4) layer propagation and terminal readouts: Eq. 16, Eq. 11-15 ----------------------------
 *   G_dev    device, fp64, read-only: G_dev[((blk*d + a)*d + b) * batch + c] = propagator of block blk
 *            from endpoint a to endpoint b (A[vbar, pi(v)bar] of Eq. 59) of configuration c;
 *            the configuration index is the contiguous one.  blk < 1 (uniform) or N_f (SB).
 *   batch    number of configurations (>= 0; 0 is a no-op).
 *   out_dev  device, fp64, written: out_dev[k*batch + c]; k = 0 for readout_envelope = 0, otherwise
 *            k = bitmask(S)-1 with bit i <-> vertex i (2^n-1 rows).
 *   stream   CUDA stream the kernels are enqueued on.  The call is asynchronous: it returns after
 *            enqueueing (launch errors only).  The handle owns the layer-slab workspace; one cos_eval in
 *            flight per handle.  After cos_reserve(h, B) every cos_eval with batch <= B only enqueues
 *            kernels (no allocation, no synchronisation: it can be captured into a CUDA graph) AS LONG AS the
 *            workspace need does not rise afterwards; without the reserve the workspace is grown on demand by a
 *            synchronising cudaFree + cudaMalloc.  The need rises with a larger batch, a larger
 *            cos_set_workspace_limit, or a change of COS_TUNE_TILES_PER_CHUNK: call cos_reserve again after any of
 *            these.  A cos_eval that would have to grow the workspace while `stream` is being captured does not
 *            allocate: it returns COS_EINVAL, enqueues nothing, and leaves the capture intact.
 *            Captured graphs hold the workspace address: a later regrowth (any of the causes above) or cos_free
 *            invalidates every graph captured from this handle -- replaying one then writes to freed memory;
 *            re-capture after cos_reserve.  cos_eval_host allocates staging buffers and synchronises: never capture it.
 * The current CUDA device must be the one the handle was built on (COS_EINVAL otherwise).
 * Large batches are processed in chunks that fit the workspace budget (cos_set_workspace_limit). */
int cos_eval(cos_handle h, const double* G_dev, long long batch, double* out_dev, cos_stream stream);

/* Allocates the layer-slab workspace for batches of up to `batch` configurations now (synchronous), under the
 * current workspace limit.  COS_ENOMEM when the device cannot hold it. */
int cos_reserve(cos_handle h, long long batch);

/* Releases host and device memory of the handle.  cos_free(NULL) is a no-op. */
void cos_free(cos_handle h);

/* Upper bound (bytes) for the layer-slab workspace of a handle; default 64 GiB. */
int cos_set_workspace_limit(cos_handle h, long long bytes);

/* Launch tuning of a handle.  These are the ONLY knobs; the library reads no environment variable (the Python binding
 * does read one, COS_B200_LIB, to pick which build of this library it loads -- nothing else).  Results do not
 * depend on them (same arithmetic, same summation order).  Bad parameter or value: COS_EINVAL. */
enum {
    COS_TUNE_PREFETCH = 0,           /* L2 look-ahead of the layer kernel, in states (0 = off; default 8) */
    COS_TUNE_WARPS_PER_CTA = 1,      /* 1..24 (what fits the handle's kernel: at most 16, or 20 for rows of 20 endpoints);
                                        default: the CTA size with the most resident warps per SM.  The handle's device
                                        must be current (COS_EINVAL otherwise) */
    COS_TUNE_BLOCKS_PER_CTA_CAP = 2, /* upper bound of occupancy-mask blocks per CTA (0 = default: one per staged table slot) */
    COS_TUNE_PDL = 3,                /* programmatic dependent launch between layers (default 1) */
    COS_TUNE_FUSED = 4,              /* small DAGs: 1 = one fused launch (default), 0 = per-layer kernels */
    COS_TUNE_HOST_SLICES = 5,        /* cos_eval_host: at most this many output slices, 1..8 (default 8; 1 = no second stream) */
    COS_TUNE_TILES_PER_CHUNK = 6     /* at most this many 32-configuration tiles per workspace chunk (0 = no bound) */
};
int cos_set_tuning(cos_handle h, int what, long long value);

/* ---- introspection (SURVEY.md section 5 "metrics") ------------------------------------------------- */
enum {
    COS_INFO_N_LAYERS = 0,        /* 2n */
    COS_INFO_N_STATES = 1,        /* DAG states over all layers (Eq. 79 keys in the reduced form of DESIGN.md) */
    COS_INFO_N_EDGES = 2,         /* DAG edges E1..E4, uncoalesced, colour fan-out included (Eq. 16) */
    COS_INFO_N_READOUT_EDGES = 3, /* sum_S q_S, Eq. 15 / PAPER.md:156 */
    COS_INFO_N_OUT = 4,           /* 1 or 2^n-1 */
    COS_INFO_MAX_LAYER_STATES = 5,
    COS_INFO_N_MASKS = 6,         /* occupancy masks (block count) */
    COS_INFO_N_ROWS = 7,          /* (mask, head, colour) rows */
    COS_INFO_N_FMA = 8,           /* fp64 FMAs the kernels execute per configuration */
    COS_INFO_PROGRAM_BYTES = 9,   /* device bytes of the compiled program */
    COS_INFO_D = 10,              /* d = n * n_sub */
    COS_INFO_N_BLOCKS = 11,       /* propagator blocks expected in G_dev */
    COS_INFO_N_STATES_UNPRUNED = 12,
    COS_INFO_WORKSPACE_BYTES = 13,
    COS_INFO_N_LAUNCHES = 14,     /* kernels launched through this handle so far (cos_eval / cos_eval_host) */
    COS_INFO_ORDER_MASK = 15,     /* requested orders of an all-subset handle (0 for single-output handles) */
    COS_INFO_RESERVED_BATCH = 16, /* largest batch passed to a successful cos_reserve so far (0: none) */
    COS_INFO_DEVICE = 19,         /* CUDA device of the handle (-1: host-only) */
    COS_INFO_FUSED = 20,          /* 1: cos_eval walks the DAG in one fused launch */
    COS_INFO_LAYER_STATES = 100,  /* + layer index */
    COS_INFO_LAYER_EDGES = 200,   /* + layer index: edges leaving that layer (readout edges included) */
    COS_INFO_LAYER_MASKS = 300    /* + layer index */
};
int cos_info(cos_handle h, int what, long long* value);

const char* cos_last_error(void);

/* ---- (2) propagator tabulation: PAPER.md:271-275 (Eq. 32), 415; readings G17-G18 of DESIGN.md --------
 * cos_tab_build copies a host lookup table to the device.
 *   table_host  host fp64, layout [n_blocks][n_sub*n_sub][L*L][n_tau]: value of g_blk^{s s'}(r, tau_k),
 *               r = (dx, dy) = displacement FROM-endpoint minus TO-endpoint modulo L, index dx*L+dy,
 *               tau_k = k*beta/(n_tau-1), k = 0..n_tau-1 (both ends).
 * cos_tabulate fills G_dev (layout of cos_eval) for `batch` configurations:
 *   A[(i,s),(j,s')] = sign * ((1-w) T[k] + w T[k+1]),  dtau = tau_i - tau_j; dtau <= 0 -> dtau += beta,
 *   sign = -1 (anti-periodicity; equal times and i = j use 0^-);  u = dtau/(beta/(n_tau-1)),
 *   k = min(floor(u), n_tau-2), w = u-k.
 *   sites_dev   device int32 [n][2][batch]   lattice (square) or unit-cell (honeycomb) coordinates in [0,L)
 *   tau_dev     device fp64  [n][batch]      imaginary times in [0, beta)
 * Times outside [0, beta) or non-finite times never cause an out-of-bounds table read: the node index is clamped to
 * [0, n_tau-2] (the value is then a linear extrapolation, or NaN for a NaN time).  Sites are reduced modulo L.
 * The current CUDA device must be the one the table was built on (COS_EINVAL otherwise).  Asynchronous on `stream`. */
int cos_tab_build(int lattice, int L, int n_blocks, double beta, int n_tau, const double* table_host, cos_tab* out);
int cos_tabulate(cos_tab tab, int n, const int* sites_dev, const double* tau_dev, long long batch,
                 double* G_dev, cos_stream stream);
void cos_tab_free(cos_tab tab);

/* ---- host-buffer pipeline: tabulate (2) + evaluate (3)+(4) for configurations that live in HOST memory.
 *   sites_host  host int32 [n][2][batch], tau_host host fp64 [n][batch] (layouts of cos_tabulate; pinned memory
 *               makes the copies asynchronous, pageable memory works too), out_host host fp64 [n_out][batch].
 * Copies the inputs to a device staging area owned by the handle (grown lazily), runs cos_tabulate and cos_eval on
 * `stream`, copies the result back and SYNCHRONISES the stream before returning.  Outputs of 16 MiB or more are
 * produced in up to 8 batch slices whose columns are copied back on an internal second stream while the next slice
 * is evaluated.  n is the handle's order; the table
 * must have the handle's number of propagator blocks and lattice.  Bytes moved per call:
 * H2D batch*n*(2*4+8), D2H batch*n_out*8. */
int cos_eval_host(cos_handle h, cos_tab tab, const int* sites_host, const double* tau_host, long long batch,
                  double* out_host, cos_stream stream);

/* ---- many-configuration heat-bath weights: Eq. 6-7 -------------------------------------
 * Phi_S = lambda_{|S|} C_S Q_S (Eq. 6),  W = sum_{S, |S| in U} |Phi_S| / binom(n, |S|) (Eq. 7), per configuration.
 *   n            envelope size N (1..COS_MAX_N)
 *   order_mask   allowed orders U (bit k <-> |S| = k); 0 = every order
 *   lambda_host  host fp64 [n+1]: lambda_k at index k (index 0 unused)
 *   C_dev        device fp64 [2^n-1][batch]: connected values, the layout cos_eval writes (k = bitmask(S)-1)
 *   Q_dev        device fp64 [2^n-1][batch] conditional densities Q_{S-bar|S}, or NULL for Q = 1
 *                (the paper takes Q from the sampler, ref. [15]; it is an input here)
 *   W_dev        device fp64 [batch], written
 *   Phi_dev      device fp64 [2^n-1][batch] signed fluxes, written (zeros outside U), or NULL to skip
 * One thread per configuration adds the subsets in increasing bitmask order (deterministic).  Asynchronous. */
int cos_flux_weights(int n, unsigned int order_mask, const double* lambda_host, const double* C_dev,
                     const double* Q_dev, long long batch, double* W_dev, double* Phi_dev, cos_stream stream);

/* ---- determinant-polynomial route on the device: PAPER.md:267-315 (Eq. 32-38); SURVEY.md 8(f).3 ---------------
 * An independent second evaluator of the all-subset connected values ("an independent comparison with SB-CoS for
 * non-uniform matrices and shifts"): principal minors d_a(S) = det A^(a)[S,S] (Eq. 34), full moments
 * H(T) = sum_{S_a} prod_a d_a(S_a) prod_i L_i with the local tensor of Eq. 35 (a site of T carries a pair of flavours
 * a < b with weight 2, or one flavour a with weight 2 sigma_a; reading G13 of DESIGN.md for two flavours), connected
 * values C(T) = H(T) - sum_{S proper subset of T, min T in S} C(S) H(T \ S) (Eq. 38; proper subsets, reading G14).
 * H has the physical convention of Eq. 83 (no shift-shift term), like cos_eval.
 *   lattice    COS_LATTICE_SQUARE (d = n), or COS_LATTICE_HONEYCOMB (d = 2n, endpoint a = 2i + s): the moments are
 *              summed over the 2^|T| sublattice labels of the vertices of T before Eq. 38 (Eq. 54-55)
 *              -- the sublattice-summed value the honeycomb DAG returns.  Implemented by walking all 2^n assignments
 *              (2^n times the square-lattice cost; every H(T) is met 2^(n-|T|) times and that power of two divided out).
 *   n_flavors  2 or 3 (COS_EUNSUPPORTED otherwise).
 *   n_blocks   n_flavors (one n x n matrix per flavour) or 1 (flavour-uniform: every flavour reads block 0; with
 *              shifts = NULL this is the uniform CoS value with loop factor N_f, Eq. 33).
 *   shifts     host, n_flavors shift-close weights sigma_a = alpha_a/U, or NULL for zero shifts.
 *   precision  COS_DET_FP64: every step in fp64.  COS_DET_DD: every step (elimination, moments, Eq. 38) in
 *              double-double arithmetic, ~106 significant bits, as the paper does for this route;
 *              inputs are the caller's fp64 values, taken as exact; outputs are rounded to fp64 at the end.
 *   G_dev      device fp64 [n_blocks][d][d][batch], the layout of cos_eval (read-only).
 *   out_dev    device fp64 [2^n-1][batch], written: row bitmask(T)-1, the layout of an all-subset cos_eval.
 *   work_dev   device scratch of at least cos_det_workspace_bytes(n, n_blocks, precision, batch) bytes, 16-byte aligned,
 *              owned by the caller; work_bytes is its size (too small or misaligned: COS_EINVAL).
 * Accuracy: Eq. 38 subtracts from H(T) every disconnected product of smaller moments, so the rounding error of the
 * route scales with R(T) = the same recursion with every term positive on |A|, |sigma| (>= the DAG's M, which has
 * only the connected terms): |error| ~ 1e-15 R in fp64, ~1e-30 R in double-double.  On physical propagators
 * |C| / R falls from ~1e-8 (n = 6) to ~1e-22 (n = 10): fp64 is a cross-check up to n ~ 6, double-double to n ~ 10-11
 * (at n = 12, beta = 8 it keeps ~5 digits of the full-order value).
 * Cost: 7^n (three flavours) or 4^n (two) terms per configuration.  Asynchronous on `stream`. */
enum { COS_DET_FP64 = 0, COS_DET_DD = 1 };
long long cos_det_workspace_bytes(int n, int n_blocks, int precision, long long batch);      /* -1 on bad arguments */
int cos_det_eval(int n, int n_flavors, int n_blocks, int lattice, const double* shifts, int precision,
                 const double* G_dev, long long batch, double* out_dev, void* work_dev, long long work_bytes,
                 cos_stream stream);

/* ---- the same route for callers that must not allocate device memory ------------------------------------------
 * cos_det_eval needs a scratch buffer, and somebody has to cudaMalloc it.  Some users of this library cannot: a
 * Monte-Carlo sampler whose steady-state loop may not contain a call that stalls the whole device (cudaMalloc and
 * cudaFree synchronise it), a plug-in running inside a host program that has already handed all free HBM to its own
 * memory pool (a further cudaMalloc simply fails there) or that forbids driver allocations in its callbacks, and
 * latency-bounded services where an allocation of unknown duration in the request path is not acceptable.
 * cos_det_eval_static is cos_det_eval with the scratch taken from an array that is compiled into the library
 * (a file-scope `static __device__` array of COS_DET_STATIC_SCRATCH_BYTES = 16 MiB): it calls neither cudaMalloc nor
 * cudaFree nor any library routine that allocates, on any call.  The caller passes inputs and outputs only.
 *   Arguments, layouts, precision, arithmetic and error codes: exactly those of cos_det_eval (same kernels, same
 *   summation order -- the results are bit-identical to cos_det_eval on the same inputs).
 *   Limit: cos_det_workspace_bytes(n, n_blocks, precision, batch) must not exceed COS_DET_STATIC_SCRATCH_BYTES, e.g.
 *   fp64 with three blocks: batch <= 1638 at n = 8, <= 409 at n = 10; double-double: half of that.  Anything larger is
 *   refused with COS_EUNSUPPORTED and a message naming both byte counts (split the batch, or use cos_det_eval with a
 *   buffer of your own); nothing is launched in that case.
 *   Cost: every GPU on which the library's CUDA code is loaded holds the 16 MiB until the process exits, used or not.
 *   Set-up: the first call on a device looks up that device's address of the array (cudaGetSymbolAddress; once per
 *   device, with the device that is current in the calling thread, remembered afterwards).  That first call may make
 *   the CUDA runtime load the library's device code, so make it during initialisation and BEFORE any stream capture
 *   is begun; later calls on that device only enqueue kernels.
 *   Sharing: there is one array per device and every call on that device uses it.  Calls are ordered correctly when
 *   they are enqueued on the same stream; two calls that can overlap on the GPU (different streams, or different host
 *   threads with their own streams) race on the scratch and return garbage -- serialise them yourself.  The array keeps
 *   whatever the previous call left in it; that is harmless here because every call writes each scratch element
 *   (minors, moments, connected values, subset order) before it reads it, so nothing has to start at zero.
 * Asynchronous on `stream`, like cos_det_eval. */
#define COS_DET_STATIC_SCRATCH_BYTES (16ll << 20)
int cos_det_eval_static(int n, int n_flavors, int n_blocks, int lattice, const double* shifts, int precision,
                        const double* G_dev, long long batch, double* out_dev, cos_stream stream);

/* ---- measurement helpers ------------------------------------------------------------------------------
 * cos_set_profiling(h, 1): every later cos_eval brackets each layer launch with CUDA events on its stream.
 * cos_get_layer_times synchronises on the recorded events, ADDS the elapsed milliseconds of layer l (summed over
 * batch chunks and over all cos_eval calls since the last cos_get_layer_times) to ms[l] for l < n_layers, stores
 * the number of profiled cos_eval calls in *n_evals, and clears the record.  ms is host memory, caller-zeroed. */
int cos_set_profiling(cos_handle h, int on);
int cos_get_layer_times(cos_handle h, int n_layers, double* ms, long long* n_evals);

/* Self-check build (libcos_b200.so compiled with -DCOS_CHECK_BOUNDS; tests/test_gpu_selfcheck.py builds one): the layer
 * kernels test every index they derive from the compiled program against the extent of the array it addresses (kinds:
 * 0 program window, 1 source row, 2 row header, 3 destination state / endpoint, 4 table row, 5 head / colour, 6 fresh-head
 * destination, 7 output row) and cos_eval fills the workspace with NaN first.  *total = violations counted so far, or -1
 * when the library was built without the checks (the shipped build); by_kind: host array of 8 counters, or NULL. */
int cos_debug_check_failures(long long* total, long long* by_kind);

/* fp64 FMA peak of the device (independent FMA chains, no memory traffic).
 * Returns achieved FMA/s in *fma_per_s (synchronous; used by bench.py for the fp64 roofline leg). */
int cos_measure_fp64_fma_peak(double* fma_per_s);

#ifdef __cplusplus
}
#endif
#endif /* COS_B200_H */
