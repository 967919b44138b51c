/*
 * gvqe.h -- C ABI of libgvqe: batched statevector VQE energy engine for NVIDIA B200 (sm_100a).
 *
 * Hot path of Graph-VQE (arxiv/paper_2607_02749; citations are lines of /root/reference/PAPER.md):
 *   |psi(theta)> = U(theta)|0>^N  for a hardware-efficient RY/RZ + CZ/CNOT ansatz   PAPER.md:169-179 (Eq. 7, 8)
 *   E(theta) = <psi|H|psi>,  H = sum_k c_k P_k,  c_k real, P_k in {I,X,Y,Z}^N        PAPER.md:135 (Eq. 4), 148-153 (Eq. 6)
 *   E = sum_j <psi|H_j|psi> over any partition of the terms ("Hamiltonian batching")  PAPER.md:214-219 (Eq. 12)
 *   restricted objective: only the block's parameters move                          PAPER.md:207-212 (Eq. 11)
 *   dE/dtheta_i = 1/2 [E(theta + pi/2 e_i) - E(theta - pi/2 e_i)]                     PAPER.md:221-225 (Eq. 13)
 *
 * Conventions: qubit q <-> bit q of the amplitude index (LSB = qubit 0); character j
 * of a Pauli string acts on qubit j; R_y, R_z exactly as Eq. 7; ops are applied in list order.
 *
 * Memory: every "host" pointer is ordinary host memory, borrowed for the duration of the call (inputs are
 * copied).  ALL device memory is the caller's workspace (gvqe_set_workspace); the library allocates none.
 * Errors: every call returns a gvqe_status; gvqe_last_error gives the message.  There is no CPU fallback:
 * a missing/failed CUDA device is GVQE_ERR_CUDA.  Results are deterministic: identical inputs give
 * bit-identical outputs (no floating-point atomics).  A context is not thread-safe.
 */
#ifndef GVQE_H
#define GVQE_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gvqe_ctx gvqe_ctx; /* opaque, owned by the library, freed by gvqe_destroy */

typedef enum {
    GVQE_OK = 0,
    GVQE_ERR_INVALID_ARG = 1,
    GVQE_ERR_NO_HAMILTONIAN = 2,
    GVQE_ERR_WORKSPACE = 3,
    GVQE_ERR_UNSUPPORTED = 4,
    GVQE_ERR_CUDA = 5
} gvqe_status;

typedef enum { GVQE_C64 = 0, GVQE_C128 = 1 } gvqe_precision;
typedef enum { GVQE_OP_RY = 0, GVQE_OP_RZ = 1, GVQE_OP_CZ = 2, GVQE_OP_CNOT = 3 } gvqe_opkind;

/* One gate.  RY/RZ: qubit q0, angle params[param], q1 = -1.  CZ: qubits q0,q1, param = -1.
 * CNOT: target q0, control q1, param = -1.  A parameter may drive at most one gate (Eq. 13 is then exact). */
typedef struct { int32_t kind, q0, q1, param; } gvqe_op;

/* Layered ansatz: for l in 0..n_layers-1: RY(theta[2Nl+q]) all q, RZ(theta[2Nl+N+q]) all q,
 * entanglers (q,q+1) ascending (CNOT: control q, target q+1), then (N-1 -> 0) if topology == 1;
 * finally RY(theta[2ND+q]) (and RZ(theta[2ND+N+q]) if final_rot == 2, which gives Eq. 8's P = 2N(D+1)). */
/* Entanglement maps (PAPER.md:260 evaluates Circular, Full, Linear, Reverse Linear, Pairwise and SCA); pairs are
 * (control, target), CZ ignores the roles.  n <= 2: every map with a wrap pair degenerates to the chain.
 *   LINEAR (q,q+1) q ascending | RING = LINEAR then (N-1,0) | FULL (i,j) all i<j, i then j ascending |
 *   REVERSE_LINEAR (q,q+1) q descending | PAIRWISE (q,q+1) even q ascending, then odd q ascending |
 *   CIRCULAR (N-1,0) then LINEAR | SCA: layer l uses the circular list C = [(N-1,0),(0,1),...,(N-2,N-1)] shifted
 *   by l places (entry j = C[(j-l) mod N]) with control and target swapped on odd l. */
typedef enum { GVQE_TOPO_LINEAR = 0, GVQE_TOPO_RING = 1, GVQE_TOPO_FULL = 2, GVQE_TOPO_REVERSE_LINEAR = 3,
               GVQE_TOPO_PAIRWISE = 4, GVQE_TOPO_CIRCULAR = 5, GVQE_TOPO_SCA = 6 } gvqe_topology;

typedef struct {
    int32_t n_layers;  /* D >= 0 */
    int32_t entangler; /* GVQE_OP_CZ or GVQE_OP_CNOT */
    int32_t topology;  /* gvqe_topology: 0 linear chain, 1 ring (chain, then the wrap pair), 2..6 see below */
    int32_t final_rot; /* 1 = RY only, 2 = RY then RZ */
} gvqe_layout;

/* Create a context (host only; touches no GPU).  1 <= n_qubits <= 34.  *out receives the context. */
gvqe_status gvqe_create(int n_qubits, const gvqe_layout *layout, gvqe_precision prec, gvqe_ctx **out);
/* Same from an explicit op list (host, n_ops entries; params are indices in [0, n_params)). */
gvqe_status gvqe_create_ops(int n_qubits, const gvqe_op *ops, int n_ops, int n_params, gvqe_precision prec,
                            gvqe_ctx **out);

/* Schedule options: HOW the same energies are computed (the circuit is compiled once and reused).  Every
 * field 0 = the library's default; results are identical up to floating-point reassociation whatever is chosen.  The
 * library reads no environment variable; tests pass these to reach every code path at small sizes. */
typedef struct {
    int32_t tile_bits;        /* k: qubits of a shared-memory tile (default 13 complex64 / 12 complex128; up to 14) */
    int32_t fixed_bits;       /* f: lowest qubits that are in every tile (default 4 / 3): 2^f contiguous amplitudes */
    int32_t reg_bits;         /* R: register bits per stage (default 5 / 4) */
    int32_t expect_tile_bits; /* tile bits of the expectation passes (default min(k, 13 / 12)) */
    int32_t prefix;           /* write-only product-state kernel for the first layer: 0 = when it saves HBM
                               * passes, 1 = never, 2 = whenever the circuit starts with a rotation layer */
    int32_t register_stages;  /* expectation: flip-mask groups evaluated from registers: 0 = on, 1 = off */
    int32_t shared_prefix;    /* gvqe_param_shift_grad: 0 = shared prefixes for states >= 16 MiB, 1 = never, 2 = always */
    int32_t specialise;       /* gate kernels generated and compiled for the schedule at the first energy call (NVRTC):
                               * 0 = for registers of >= 20 qubits when NVRTC is present, 1 = never (generic kernels),
                               * 2 = whenever the schedule is supported; GVQE_ERR_UNSUPPORTED at the first energy call if
                               * it is not or NVRTC is missing */
    int32_t tiles_per_block;  /* specialised kernels: consecutive tiles one thread block works through (its per-block
                               * set-up is paid once): 0 = default (tuned on the B200), else 1..4096 */
    int32_t blocks_per_sm;    /* specialised gate kernels: thread blocks resident per SM the kernels are compiled for
                               * (register budget 65536 / (256 * blocks_per_sm)): 0 = default, else 2 or 3 */
    int32_t staged_io;        /* specialised gate kernels: 0 = the first / last stage of a block exchanges its amplitudes with
                               * global memory directly when it carries no CNOT run, 1 = every tile is staged in shared memory */
    int32_t mid_cnot;         /* specialised gate kernels: 0 = a CNOT whose target is a register qubit of its stage is applied in
                               * registers and rotations may follow it in the same stage (fewer stages), 1 = every CNOT is
                               * part of a stage's trailing run (the generic kernels' schedule) */
    int32_t interleave;       /* specialised gate kernels: thread blocks in groups of this many (a power of two <= 1024) take
                               * neighbouring tiles at the same time: 0 = default (32, tuned on the B200), 1 = consecutive tiles per
                               * thread block */
    int32_t reserved[3];      /* must be 0 */
} gvqe_options;
/* gvqe_create / gvqe_create_ops with options (opt == NULL: defaults). */
gvqe_status gvqe_create_opt(int n_qubits, const gvqe_layout *layout, gvqe_precision prec, const gvqe_options *opt,
                            gvqe_ctx **out);
gvqe_status gvqe_create_ops_opt(int n_qubits, const gvqe_op *ops, int n_ops, int n_params, gvqe_precision prec,
                                const gvqe_options *opt, gvqe_ctx **out);
/* Source text of specialised kernel number `block` as the library would compile it: the fused gate blocks first
 * (0-based, in execution order), then -- once a Hamiltonian is set -- the expectation passes; written to
 * buf (NUL-terminated, truncated to cap); returns the full length needed, 0 when there is no such kernel.
 * *smem_bytes (optional): its dynamic shared memory.  Host only (no GPU, no compiler). */
size_t gvqe_kernel_source(const gvqe_ctx *ctx, int block, char *buf, size_t cap, int32_t *smem_bytes);
/* Facts about specialised kernel number `block` (numbering as gvqe_kernel_source): out[0] = 0 gate block / 1 expectation
 * pass, out[1] = dynamic shared memory in bytes, out[2] = floating-point lane operations per amplitude and launch the
 * schedule needs (2 per rotation in tangent form, 4 per complex phase factor, 6 / 4 / 3 per amplitude pair of a
 * complex / real / imaginary W): the numerator of the ALU roofline, out[3] = 0.  GVQE_ERR_INVALID_ARG if no such kernel. */
gvqe_status gvqe_kernel_info(const gvqe_ctx *ctx, int block, double *out);
/* The arrays the specialised expectation kernels read from global memory, as host images (introspection for tests):
 * which = 0: static W tables (double re, im per entry), 1: tile-dependent index patterns (4 x uint32: shared-memory byte
 * offset, first term, last term + 1, 0), 2: terms (double re, im of c_k i^{nY}; uint64 z bits outside the tile; uint64
 * local z mask for direct groups), 3: per pass (uint32 first table entry, first pattern, number of patterns).
 * Copies min(cap, size) bytes into buf; returns the size in bytes (0: no specialised expectation kernels). */
size_t gvqe_kernel_arrays(const gvqe_ctx *ctx, int which, void *buf, size_t cap);
/* Compiles every specialised kernel of the context with NVRTC for sm_100a (host only: needs the compiler library, no
 * GPU; images are cached for the first energy call).  *n_kernels (optional): how many were compiled (0 when the
 * context uses the generic kernels).  GVQE_ERR_UNSUPPORTED with the compiler's message when NVRTC is missing or a
 * kernel does not compile.  Used by the build check. */
gvqe_status gvqe_compile_kernels(gvqe_ctx *ctx, int32_t *n_kernels);
int gvqe_num_params(const gvqe_ctx *ctx);
int gvqe_num_qubits(const gvqe_ctx *ctx);

/* Hamiltonian, Eq. 6.  paulis: host, n_terms * n_qubits characters of "IXYZ" (no separators, character j of a
 * term acts on qubit j); coeffs: host, n_terms finite doubles.  Identity and duplicate terms are legal.
 * Host work only (parse -> masks -> flip-mask groups); device tables are (re)built on the next energy call. */
gvqe_status gvqe_set_hamiltonian(gvqe_ctx *ctx, int n_terms, const char *paulis, const double *coeffs);
/* Same from masks: x_mask = qubits with X or Y, z_mask = qubits with Z or Y (so Y = both bits). */
gvqe_status gvqe_set_hamiltonian_masks(gvqe_ctx *ctx, int n_terms, const uint64_t *x_mask, const uint64_t *z_mask,
                                       const double *coeffs);
/* Integer side of the grouping (bit-exact contract): per term x_mask, z_mask, n_Y mod 4, group index; groups are
 * the distinct x_mask values in ascending unsigned order (group_mask[g]).  Output arrays are host, caller-owned,
 * sized n_terms (group_mask: n_terms is always enough); any may be NULL. */
gvqe_status gvqe_get_grouping(const gvqe_ctx *ctx, uint64_t *x_mask, uint64_t *z_mask, uint8_t *ny_mod4,
                              int32_t *group_of_term, int32_t *n_groups, uint64_t *group_mask);

/* Device workspace.  gvqe_workspace_bytes: bytes needed to keep `batch_in_flight` statevectors resident (plus
 * tables and scratch); 0 on error.  Call after gvqe_set_hamiltonian.  gvqe_set_workspace: device_ptr is DEVICE
 * memory (256-byte aligned) owned by the caller, which must stay valid until gvqe_destroy or the next
 * gvqe_set_workspace; too small for one statevector -> GVQE_ERR_WORKSPACE.  Larger batches are streamed in
 * chunks of as many statevectors as fit (at most max_in_flight if that was set > 0). */
size_t gvqe_workspace_bytes(const gvqe_ctx *ctx, int batch_in_flight);
gvqe_status gvqe_set_workspace(gvqe_ctx *ctx, void *device_ptr, size_t bytes);
gvqe_status gvqe_set_max_in_flight(gvqe_ctx *ctx, int max_in_flight);

/* E[b] = <psi(params[b])|H|psi(params[b])>, Eq. 4.  params: HOST, B x P row-major doubles (finite); E: HOST, B
 * doubles.  cuda_stream: a cudaStream_t (NULL = default stream).  Returns after E is on the host. */
gvqe_status gvqe_energy_batch(gvqe_ctx *ctx, const double *params, int B, double *E, void *cuda_stream);
/* Same with DEVICE pointers (params_dev: B x P doubles, E_dev: B doubles); asynchronous on the stream, no host
 * copies or synchronisation.  This is the entry the device-resident timing uses. */
gvqe_status gvqe_energy_batch_device(gvqe_ctx *ctx, const double *params_dev, int B, double *E_dev, void *cuda_stream);

/* Eq. 13 over the parameters with mask[p] != 0 (Eq. 11: the cluster's parameters).  params: HOST, P doubles;
 * mask: HOST, P bytes; dE: HOST, P doubles (0 where mask is 0); E0: HOST, optional (NULL allowed), receives
 * E(params).  The 2|mask|+1 evaluations run as one batch (row 0 = theta, rows 2j+1 / 2j+2 = +/- pi/2 on the
 * j-th masked parameter).  With more than one statevector in flight and states of at least 16 MiB (smaller ones are
 * launch-bound; gvqe_options.shared_prefix overrides) the rows are evaluated with shared prefixes: the
 * state of theta advances block by block and a shifted row starts from the boundary at which its parameter is first
 * read; the results are bit-identical to gvqe_energy_batch on the expanded rows. */
gvqe_status gvqe_param_shift_grad(gvqe_ctx *ctx, const double *params, const uint8_t *mask, double *dE, double *E0,
                                  void *cuda_stream);

/* Test hook: amplitudes (interleaved re,im in the context's precision, 2^n of them) of in-flight slot `slot`
 * as left by the last energy call, copied to host_out (HOST). */
gvqe_status gvqe_get_state(gvqe_ctx *ctx, int slot, void *host_out);

/* Read-out, PAPER.md:245 ("the bitstring with the highest probability is identified as the optimal turn sequence"):
 * *x = argmax_x |psi_x|^2 over the statevector in in-flight slot `slot` as left by the last energy call (bit q of
 * x = qubit q), ties to the lowest x; *prob (HOST, optional) = that probability.  |psi_x|^2 = re*re + im*im in the
 * context's precision, each operation rounded separately.  One read-only sweep of the state on the GPU. */
gvqe_status gvqe_argmax(gvqe_ctx *ctx, int slot, uint64_t *x, double *prob, void *cuda_stream);

/* The same read-out for callers that may not allocate device memory -- code under CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc.  Needs no context and no workspace; calls no cudaMalloc / cudaFree or
 * any allocating routine, copies nothing to the host and does not synchronise: two kernel launches on cuda_stream.
 *   state         DEVICE, n_amplitudes complex numbers (interleaved re, im) of precision prec, 16-byte aligned; read only
 *   n_amplitudes  1 .. GVQE_NOALLOC_MAX_AMPLITUDES (2^34); anything else is GVQE_ERR_INVALID_ARG
 *   result        DEVICE, 16 bytes, 8-byte aligned, written by the call: { double prob; uint64_t x; } with the meaning, tie
 *                 rule and arithmetic of gvqe_argmax (bit-identical to it on the same amplitudes)
 *   err, err_cap  HOST, optional: receives the message of a failed call (NUL-terminated, truncated to err_cap)
 * Scratch: the per-block candidates live in a file-scope device array of GVQE_NOALLOC_SCRATCH_BYTES (32 KiB) that every
 * GPU which loads the library holds until the process exits.  All calls on a device share it and it keeps the last
 * call's contents (none of which a later call reads): calls that overlap on the GPU -- different streams without an
 * ordering between them -- race on it; calls on one stream, or ordered by events, are safe.  The first call on a device
 * looks the array's address up (cudaGetSymbolAddress); make that call before a graph capture starts. */
#define GVQE_NOALLOC_MAX_AMPLITUDES (1ull << 34)
#define GVQE_NOALLOC_SCRATCH_BYTES (32u * 1024u)
gvqe_status gvqe_argmax_noalloc(const void *state, uint64_t n_amplitudes, gvqe_precision prec, void *result,
                                void *cuda_stream, char *err, size_t err_cap);

/* Shot sampling, PAPER.md:245, 256 ("this state is sampled"; 8192 shots): n_shots (<= 65536 per call) bitstrings
 * distributed as |psi_x|^2 over the state in slot `slot`, by inversion of the cumulative distribution in index
 * order: x[s] = the first x with sum_{y<=x} |psi_y|^2 > u[s] * Z, Z = sum_y |psi_y|^2.  The random numbers are the
 * caller's: u: HOST, n_shots doubles in [0,1); x: HOST, n_shots results; *norm (HOST, optional) = Z.  Sums are fp64 in
 * a fixed order (deterministic); a shot whose u * Z falls within rounding of a cumulative boundary may land on
 * either neighbour. */
gvqe_status gvqe_sample(gvqe_ctx *ctx, int slot, int n_shots, const double *u, uint64_t *x, double *norm,
                        void *cuda_stream);

/* Finite-shot energy estimate, PAPER.md:256 ("8192 measurement shots" per evaluation), 270 (shot-noise study).
 * Measurement settings (reading R3): two terms share a setting when they carry the same X / Y letters on the same
 * qubits; settings are numbered in ascending (x_mask, y_mask) order (Z-only and identity terms: setting 0 when present).
 * gvqe_measurement_settings: *n_settings and, per term (HOST, n_terms entries, may be NULL), its setting.
 * gvqe_energy_shots: for every setting the statevector of in-flight slot `slot` (as left by the last energy call) is
 * copied into another slot, rotated into the setting's basis (H on the X qubits, H S^dagger on the Y qubits), n_shots
 * bitstrings are drawn by inversion exactly as in gvqe_sample with the caller's uniforms u[setting * n_shots + s]
 * (HOST, n_settings * n_shots doubles in [0,1)), and <P_k> is estimated as the mean of (-1)^{popcount(x & support_k)} over
 * the shots of the term's setting.  *E_est = sum_k c_k <P_k>_est; term_means (HOST, optional, n_terms doubles).  Needs at
 * least two statevectors in flight (GVQE_ERR_WORKSPACE otherwise); n_shots <= 65536.  The slot's own state is unchanged. */
gvqe_status gvqe_measurement_settings(const gvqe_ctx *ctx, int32_t *n_settings, int32_t *setting_of_term);
gvqe_status gvqe_energy_shots(gvqe_ctx *ctx, int slot, int n_shots, const double *u, double *E_est, double *term_means,
                              void *cuda_stream);

/* Introspection of the compiled schedule (host; for tests and traffic accounting).
 * gvqe_schedule_info: number of fused gate blocks, number of off-diagonal passes, statevectors in flight.
 * gvqe_dump_schedule: writes a text description of every block/stage/op into buf (NUL-terminated, truncated to
 * cap); returns the full length needed. */
gvqe_status gvqe_schedule_info(const gvqe_ctx *ctx, int32_t *n_gate_blocks, int32_t *n_offdiag_passes,
                               int32_t *in_flight);
size_t gvqe_dump_schedule(const gvqe_ctx *ctx, char *buf, size_t cap);
/* The order in which the device executes the input ops (indices into the op list, each exactly once; the
 * compiler only reorders ops that commute).  order: host, cap entries; returns the number of ops. */
int gvqe_get_exec_order(const gvqe_ctx *ctx, int32_t *order, int cap);
/* Kernel launches issued by this context since creation (for bench.py's gpu_launches). */
uint64_t gvqe_launch_count(const gvqe_ctx *ctx);

/* Per-phase device timing (CUDA events on the caller's stream around the gate blocks and around the expectation
 * passes of every chunk).  gvqe_profile_enable(ctx, 1) resets the counters and starts recording, (ctx, 0) stops.
 * gvqe_profile_read synchronises the recorded events and fills out[8] (host):
 *   [0] gate-block kernel time, ms      [1] gate-block launches   [2] gate-block algorithmic bytes (SURVEY 8(d):
 *   2*S per block and state, S for the write-only first block)     [3] expectation-pass kernel time, ms
 *   [4] expectation-pass launches       [5] expectation algorithmic bytes (S per pass and state + the table once
 *   per launch of the pass that carries the diagonal part)         [6] other kernels (expand, reduce) time, ms
 *   [7] chunks recorded. */
gvqe_status gvqe_profile_enable(gvqe_ctx *ctx, int on);
gvqe_status gvqe_profile_read(gvqe_ctx *ctx, double *out);
/* Per-launch device times of the recorded chunks, in execution order: [product-state kernel if the schedule has one],
 * fused gate blocks, expectation passes.  mean_ms / min_ms / max_ms: HOST, cap doubles each (any may be NULL); returns
 * the number of launches per chunk (-1 on a NULL context).  The spread between chunks is what min / max show. */
int gvqe_profile_read_launches(gvqe_ctx *ctx, double *mean_ms, double *min_ms, double *max_ms, int cap);

/* ---- Host-side Graph-VQE driver (north_star item 3: partitioning and the optimiser loop stay on the host as plain
 * C++).  These calls do no GPU work of their own; gvqe_graph_vqe_minimize obtains every energy and gradient through
 * gvqe_energy_batch / gvqe_param_shift_grad above.  All pointers are HOST memory owned by the caller. ---------------- */

/* Eq. 9: w[i*n+j] = sum of |c_k| over the terms that act non-trivially on both qubit i and
 * qubit j (i != j); symmetric, zero diagonal.  w: n*n doubles (n = gvqe_num_qubits).  Needs a Hamiltonian. */
gvqe_status gvqe_interaction_graph(const gvqe_ctx *ctx, double *w);
/* Eq. 10 with a resolution factor gamma on the null-model term (gamma = 1: the paper's Q):
 * Q = 1/(2m) sum_ij [w_ij - gamma k_i k_j / (2m)] delta(c_i, c_j).  community: n labels >= 0.  Q = 0 if m = 0. */
gvqe_status gvqe_modularity(int n, const double *w, const int32_t *community, double gamma, double *Q);
/* Louvain community detection on w: local moving in ascending qubit order (a qubit moves to the
 * neighbouring community of largest modularity gain; ties: stay, else the lowest label), then aggregation,
 * repeated until a level moves nothing.  community: n labels out, 0..K-1 in order of first appearance by ascending
 * qubit; *n_communities = K; *Q (optional) = Eq. 10 of the result.  Deterministic. */
gvqe_status gvqe_louvain(int n, const double *w, double gamma, int32_t *community, int32_t *n_communities, double *Q);
/* PAPER.md:197 ("blocks smaller than S_min are iteratively merged with neighbors"): while a block has fewer than
 * s_min qubits, the smallest such block (ties: lowest label) joins the block it shares the largest total weight
 * with (ties: lowest label).  community: in/out, relabelled by first appearance; *n_communities = new K. */
gvqe_status gvqe_merge_small_blocks(int n, const double *w, int s_min, int32_t *community, int32_t *n_communities);
/* The comparison partition of PAPER.md:229 ("geometric alternating offsets"): consecutive qubits in blocks of
 * block_size, the block boundaries shifted by offset (0 <= offset < block_size): qubits [0, offset) form the first
 * block when offset > 0, then [offset, offset + block_size), ...  Alternating the offset between epochs (e.g. 0 and
 * block_size / 2) is the caller's loop.  community: n labels out, *n_communities = K. */
gvqe_status gvqe_geometric_blocks(int n, int block_size, int offset, int32_t *community, int32_t *n_communities);
/* theta_{B_i} (reading A11): mask[p] = 1 when parameter p drives a rotation on a qubit q with
 * community[q] == block, else 0.  mask: P bytes. */
gvqe_status gvqe_block_param_mask(const gvqe_ctx *ctx, const int32_t *community, int32_t block, uint8_t *mask);

typedef struct {
    int32_t max_epochs;     /* >= 1 */
    int32_t block_iters;    /* L-BFGS iterations per block and epoch (0 = skip the block phase) */
    int32_t global_iters;   /* iterations of the global refinement per epoch (0 = the paper's no_Global ablation) */
    int32_t window;         /* W of Eq. 14 (paper: 40) */
    int32_t patience;       /* p_block = p_global of Eq. 14 (paper: 12) */
    int32_t epoch_patience; /* p_epoch (paper: 3) */
    int32_t lbfgs_memory;   /* correction pairs kept (>= 1) */
    int32_t optimizer;      /* PAPER.md:221 "both derivative-free (COBYLA) and gradient-based (L-BFGS-B)": 0 = L-BFGS on
                             * parameter-shift gradients, 1 = COBYLA (linear-approximation simplex method, no gradients;
                             * block_iters / global_iters then bound the energy evaluations after the first simplex) */
    double tol;             /* eps_tol of Eq. 14 and the epoch-level improvement threshold (paper: 1e-4); also COBYLA's
                             * final trust-region radius rho_end (SciPy's tol) */
    double f_tol;           /* L-BFGS relative decrease tolerance; g_tol = 0.1 f_tol */
    double rho_beg;         /* COBYLA: first trust-region radius in radians; 0 = 1.0 (SciPy's default rhobeg) */
} gvqe_opt_options;

typedef struct {
    double E_best;          /* best energy found; params holds the matching vector */
    int64_t energy_evals;   /* circuit-energy evaluations issued (rows of all batches) */
    int32_t epochs, n_blocks, steps /* accepted L-BFGS steps */, stop_reason /* 0 max_epochs, 1 epoch patience */;
} gvqe_opt_result;

/* Graph-VQE epochs: from theta*_best, every block minimises Eq. 11 over its own parameters
 * (L-BFGS on parameter-shift gradients, Eq. 13, or COBYLA: opt->optimizer) starting from the same vector, the block solutions are fused, a
 * global refinement over all parameters follows, the best vector is kept, and the run stops after epoch_patience
 * epochs without an improvement larger than tol.  Blocks run one after another on this GPU (the paper's worker
 * pool is out of scope).  params: P doubles in/out; history (optional): energy before the first epoch and after
 * every epoch, at most history_cap entries, *history_len written. */
gvqe_status gvqe_graph_vqe_minimize(gvqe_ctx *ctx, const gvqe_opt_options *opt, const int32_t *community,
                                    double *params, gvqe_opt_result *result, double *history, int32_t history_cap,
                                    int32_t *history_len, void *cuda_stream);

/* The derivative-free minimiser of the loop above on a caller-supplied function (HOST only, no GPU; used by the CPU
 * tests to compare it with SciPy's COBYLA): minimises f over x (n doubles, in/out).  f(rows, B, out, user) receives B
 * points of n coordinates (row-major, HOST) and writes out[B]; a non-zero return aborts.  rho_beg >= rho_end > 0: first
 * and last trust-region radius; max_evals: evaluation budget.  *f_best (optional) = f at the returned x; counts
 * (optional, 6 x int32): evaluations, trust-region steps, geometry steps, radius reductions, simplex rebuilds,
 * improving steps.  *reason (optional): 0 = rho_end reached, 1 = evaluation budget.  The method: PAPER.md:214, 221 name
 * COBYLA; Powell's linear-approximation method without constraints, see csrc/cobyla.cpp. */
typedef int (*gvqe_batch_fn)(const double *rows, int32_t n_rows, double *out, void *user);
gvqe_status gvqe_cobyla_minimize(int32_t n, double *x, double rho_beg, double rho_end, int32_t max_evals, gvqe_batch_fn f,
                                 void *user, double *f_best, int32_t *counts, int32_t *reason);

const char *gvqe_last_error(const gvqe_ctx *ctx);
void gvqe_destroy(gvqe_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* GVQE_H */
