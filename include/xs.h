/*
 * xs.h -- C ABI of the B200 quasi-greedy clone-sweep library (libxs_b200.so).
 *
 * What the library computes (PAPER.md = text of arXiv 2102.09510; line numbers cited):
 *   the quasi-greedy (QG) local search of PAPER.md L65-L71 / L101 run on many "clones"
 *   (L73-L85) of the diluted 3-spin model H = -sum_{(i,j,k) in E} J_ijk s_i s_j s_k on a
 *   random 3-regular 3-uniform hypergraph (L41 Eq.(1)), clones bit-packed as multi-spin
 *   coded words (L87), swept set by set over independent sets of spins (L277-L289), with
 *   the exact sweep of the first ground-state hit recorded per clone (L293) and the run's
 *   time-to-solution TTS = min over clones (L111).  DESIGN.md lists every reading taken
 *   where the paper is silent (noise granularity, Philox counters, order, stop rule).
 *
 * Conventions
 *   - Everything is integer / Boolean; there is no floating point on the path except in
 *     the small host statistics of xs_tts_stats.
 *   - "dev" pointers are CUDA device pointers owned by the caller (e.g. torch tensors'
 *     data_ptr()); "host" pointers are ordinary host memory.  The library never allocates
 *     device memory and never creates streams.  `cuda_stream` is a cudaStream_t passed as
 *     void* (NULL = the legacy default stream).
 *   - State layout: x[inst][i][w], uint64, i = spin 0..N-1, w = word 0..W-1; bit b of word w
 *     is clone c = 64 w + b; bit value 1 <=> s_i = -1.  (SURVEY.md section 8(a).)
 *   - Sweep index t is 1-based and global per instance: a call continues where the previous
 *     one stopped.  first_hit[inst][c] = t of the first sweep after which clone c has
 *     E = -N (0 if the initial state already has; XS_NO_HIT = never so far).
 *   - Every call returns 0 (XS_OK) or a negative error code; nothing throws or aborts across
 *     the ABI; xs_last_error() returns a thread-local description of the last failure.
 *   - A batch lives on the CUDA device that is current when it is created; every later call on it
 *     must be made with that device current and a stream of that device (the Python binding's
 *     Batch does this for the caller).
 *   - All calls that take a stream only enqueue work on it; xs_tts also synchronises it.
 *     xs_create_instance* additionally block the host until the table uploads are done.
 */
#ifndef XS_H_
#define XS_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define XS_OK       0
#define XS_EINVAL  -1   /* null pointer, bad shape (N < 3, W = 0, n_instances = 0), bad array contents */
#define XS_ENOMEM  -2   /* caller's workspace too small / host allocation failed                        */
#define XS_ECUDA   -3   /* a CUDA runtime call or kernel launch failed                                   */
#define XS_ESTATE  -4   /* call order / handle misuse (e.g. sweep counter would overflow)                */

#define XS_NO_HIT  0xFFFFFFFFu

/* xs_params.flags */
#define XS_FLAG_GAUGE        1u  /* planted gauge: J_t = tau_i tau_j tau_k (BASELINE.json configs);
                                    off => J = +1, the paper's ferromagnet (L43)                        */
#define XS_FLAG_NO_SKIP      2u  /* keep sweeping instances that already have a solved clone
                                    (config 2: fixed sweep count).  Default: an instance whose solved
                                    flag is set at call entry is skipped (L129/L293 stop rule)          */
#define XS_FLAG_STREAMING    4u  /* force the streaming (global-memory) regime even if a tile fits
                                    on chip; the regimes are bit-identical (tests use this)             */
#define XS_FLAG_BALANCED     8u  /* generated instances: balanced independent sets instead of the
                                    greedy ones (L281: sets sized to keep the lanes evenly busy).
                                    q = max(4, ceil(N/S)) sets of equal size (within one), S = set_cap
                                    or by default the largest of 16..256 (powers of two) <= N/4,
                                    found by a deterministic tabu search seeded by
                                    the graph seed (DESIGN.md R-balance); N > 8192 or a failed search:
                                    the greedy sets.  A different, equally valid update order:
                                    trajectories differ from the greedy order's                         */
#define XS_FLAG_CLONE_NOISE 16u  /* every clone draws its own random number
                                    instead of one per word (L87): for spin i, word w, sweep t, clone
                                    bit b, U = 7-bit number whose bit k is bit b of r_k, r_2j = o0|o1<<32,
                                    r_2j+1 = o2|o3<<32 of Philox(ctr=(i,4w+j,t,6), key=run seed), j=0..3;
                                    a k = 1 spin flips iff U < m, m = round(w1_threshold / 2^25)
                                    (default: 7, w1 = 7/128).  Runs on the clause-word kernel when the
                                    batch has balanced sets that fill the CTA, else in the streaming
                                    regime; only the quasi-greedy form of the flip table is accepted   */

/* w1 = 0.055 (L101) as a 32-bit threshold: flip a k=1 spin iff u32 < floor(0.055 * 2^32). */
#define XS_W1_THRESHOLD_DEFAULT 236223201u

typedef struct xs_batch xs_batch;       /* opaque: >= 1 instances of equal N and W */

typedef struct {
    uint32_t n_spins;        /* N: spins = triplets per instance (L43), >= 3                     */
    uint32_t n_words;        /* W: uint64 words per spin; 64 W clones per instance (L87), >= 1   */
    uint32_t n_instances;    /* >= 1                                                             */
    uint32_t set_cap;        /* cap on independent-set size; 0 = uncapped (paper: 32, L279)      */
    uint32_t w1_threshold;   /* see XS_W1_THRESHOLD_DEFAULT                                      */
    uint32_t flags;          /* XS_FLAG_*                                                        */
} xs_params;

typedef struct {
    uint32_t solved;         /* 1 iff some clone of the instance has first_hit != XS_NO_HIT      */
    uint32_t tts_sweeps;     /* min_c first_hit (L111), XS_NO_HIT if not solved                  */
    uint32_t clone;          /* smallest clone index attaining the minimum, XS_NO_HIT if none    */
    uint32_t _pad;
    uint64_t sweeps_done;    /* sweeps performed on this instance so far                         */
} xs_tts_rec;

/* Host-side description of the launch geometry chosen for a batch (for bench / roofline). */
typedef struct {
    uint32_t regime;         /* 0 = on-chip tile kernel, 1 = streaming kernel                    */
    uint32_t tile_words;     /* T: uint64 columns per CTA tile (on-chip), W (streaming)          */
    uint32_t threads;        /* threads per CTA                                                  */
    uint32_t ctas;           /* CTAs per xs_run_sweeps launch                                    */
    uint32_t smem_bytes;     /* dynamic shared memory per CTA                                    */
    uint32_t batch_sweeps;   /* sweeps between ground-state checks inside the kernel             */
    uint32_t n_sets_max;     /* largest number of independent sets over the instances            */
    uint32_t variant;        /* on-chip: 0 = generic tile kernel, 1 = static-task (spin-word)
                                kernel, 2 = clause-word kernel, 3 = latency kernel (W <= 4 words:
                                one consumer warp per word + noise producer warps)               */
} xs_layout;

/* Explicit launch geometry (xs_set_geometry).  Every field is a request: 0 (XS_GEOM_AUTO for
 * `variant`) leaves the choice to the library's rule (DESIGN.md section 7 "Geometry rule"); a
 * request the shape cannot satisfy (e.g. a tile that does not fit in shared memory, a kernel
 * that does not take the update order) falls back to the rule for that field, and
 * xs_get_layout reports what was chosen.  All geometries give bit-identical results. */
#define XS_GEOM_AUTO 0xFFFFFFFFu
typedef struct {
    uint32_t variant;        /* XS_GEOM_AUTO or the on-chip kernel to prefer (xs_layout.variant)  */
    uint32_t tile_words;     /* T: 1, 2, 4, ... 64 uint64 columns per CTA tile                    */
    uint32_t threads;        /* threads per CTA, multiple of 32, <= 1024                          */
    uint32_t words_per_lane; /* static-task kernel: 1 or 2 uint64 words per lane                  */
    uint32_t batch_sweeps;   /* sweeps between in-kernel ground-state checks (>= 1)               */
    uint32_t noise_sweeps;   /* generic kernel: sweeps of noise bytes produced at a time (>= 1)   */
} xs_geometry;

/* Bytes of device workspace a batch with these parameters needs (state, first-hit table,
 * graph tables, per-instance records).  Host call, no CUDA work. */
int xs_workspace_bytes(const xs_params* p, size_t* device_bytes);

/* a-1 + a-2 of DESIGN.md.  Builds n_instances instances on the host from graph_seeds[inst]
 * (configuration model with rejection, planted gauge, adjacency, greedy independent sets;
 * DESIGN.md section "Readings"), uploads the tables into dev_ws (caller-owned, at least
 * xs_workspace_bytes, 256-byte aligned), and enqueues the init kernel that writes the random
 * initial clone states from Philox(run_seeds[inst]) (L77) and marks clones that start in a
 * ground state.  graph_seeds / run_seeds: host arrays [n_instances].  The handle owns only
 * host metadata; free it with xs_destroy.  The workspace must outlive the handle. */
int xs_create_instance(xs_batch** out, const xs_params* p, const uint64_t* graph_seeds,
                       const uint64_t* run_seeds, void* dev_ws, size_t ws_bytes,
                       void* cuda_stream);

/* Same, but the instances are given explicitly (host arrays):
 *   tri      [inst][N][3]  spin indices of each triplet (each spin in exactly 3, distinct in a triplet)
 *   jbit     [inst][N]     1 <=> J_t = -1
 *   order    [inst][N]     update order: concatenation of the independent sets (L289)
 *   set_size [inst][n_sets_max] sizes of the sets, zero padded; n_sets[inst] = number used.
 * Every set must be an anti-clique (L277); violations give XS_EINVAL. */
int xs_create_instance_from_arrays(xs_batch** out, const xs_params* p, const uint32_t* tri,
                                   const uint8_t* jbit, const uint32_t* order,
                                   const uint32_t* set_size, const uint32_t* n_sets,
                                   uint32_t n_sets_max, const uint64_t* run_seeds,
                                   void* dev_ws, size_t ws_bytes, void* cuda_stream);

/* a-3 .. a-10 (+ the termination part of a-11).  Advances every instance that is not
 * skipped (see XS_FLAG_NO_SKIP) by exactly n_sweeps sweeps (L65-L67 rule, L87 one random
 * number per word, L277 set by set), keeps first_hit exact, then refreshes the
 * per-instance solved / TTS records on the device.  Asynchronous on cuda_stream. */
int xs_run_sweeps(xs_batch* b, uint64_t n_sweeps, void* cuda_stream);

/* general flip table.  PAPER.md L67: w_k = probability of flipping a spin
 * that enters k unsatisfied interactions; the quasi-greedy rule is w = (0, 0.055, 1, 1); L69:
 * w0 = w1^3, w2 = w3 = 1 satisfies detailed balance (Metropolis at T = -2 / ln w1).
 * thr4[k] in [0, 2^32] (host array): the spin flips iff the word's 32-bit number u < thr4[k];
 * the same u serves every k (L87).  Takes effect from the next xs_run_sweeps; the default after
 * xs_create_instance* is (0, w1_threshold, 2^32, 2^32).  The quasi-greedy form and, on balanced
 * sets that fill the CTA, the family (w0, w1, 1, 1) with 0 < w0 <= w1 (Metropolis) run on the
 * clause-word kernel; other tables on the generic / streaming kernels; with thr4[0] > 0 a ground state can be left
 * again, so first hits are looked for after every sweep.  The launch geometry is chosen anew
 * (a table can move the batch to another kernel); tables a kernel needs are uploaded on
 * cuda_stream, which is synchronised if an upload happens. */
int xs_set_flip_table(xs_batch* b, const uint64_t* thr4, void* cuda_stream);

/* Overrides the automatic launch geometry (see xs_geometry); g = NULL restores the rule.
 * XS_EINVAL for malformed requests (tile_words not a power of two <= 64, threads not a multiple
 * of 32 or > 1024, words_per_lane > 2).  Takes effect from the next xs_run_sweeps; uploads kernel
 * tables on cuda_stream like xs_set_flip_table. */
int xs_set_geometry(xs_batch* b, const xs_geometry* g, void* cuda_stream);

/* a-11.  E_c = -sum_t J_t s_i s_j s_k (L41) for every clone: dev_out [inst][64 W] int32. */
int xs_energy(xs_batch* b, int32_t* dev_out, void* cuda_stream);

/* a-11/a-12.  Copies the per-instance records to host_out [n_instances] and synchronises
 * cuda_stream. */
int xs_tts(xs_batch* b, xs_tts_rec* host_out, void* cuda_stream);

/* State access (device to device, async).  xs_set_spins also recomputes first_hit from
 * scratch for the new state (clones in a ground state get the current sweep count) and
 * clears the solved flags accordingly; the sweep counters are unchanged. */
int xs_get_spins(xs_batch* b, uint64_t* dev_out /* [inst][N][W] */, void* cuda_stream);
int xs_set_spins(xs_batch* b, const uint64_t* dev_in /* [inst][N][W] */, void* cuda_stream);
int xs_get_first_hit(xs_batch* b, uint32_t* dev_out /* [inst][64 W] */, void* cuda_stream);

/* Host copies of instance `inst`'s graph: tri [N][3], jbit [N], order [N], set_size [N]
 * (first *n_sets entries valid).  Any pointer may be NULL.  No CUDA work. */
int xs_get_graph(const xs_batch* b, uint32_t inst, uint32_t* tri, uint8_t* jbit,
                 uint32_t* order, uint32_t* set_size, uint32_t* n_sets);

/* a-1 alone, host only (no CUDA work): builds one instance from graph_seed exactly as
 * xs_create_instance does and writes tri [N][3], jbit [N], order [N], set_size [N] (first
 * *n_sets entries valid), *attempt = index of the accepted configuration-model attempt.
 * Any output pointer may be NULL.  flags: only XS_FLAG_GAUGE and XS_FLAG_BALANCED are looked at. */
int xs_generate_graph(uint32_t n_spins, uint64_t graph_seed, uint32_t flags, uint32_t set_cap,
                      uint32_t* tri, uint8_t* jbit, uint32_t* order, uint32_t* set_size,
                      uint32_t* n_sets, int32_t* attempt);

/* Host only (no CUDA work): the shared-memory placement the clause-word kernel uses for the
 * instance xs_generate_graph builds from the same arguments.  The kernel keeps one
 * 64-byte row per interaction t, c_t = x_i ^ x_j ^ x_k ^ J_t (a spin's update
 * needs only the number of unsatisfied interactions it enters), in the lower or upper half of
 * 128-byte line t.  A sweep is *n_rounds rounds (>= 4, <= 16); a round puts one spin on each of the
 * CTA's n_slots slots; an independent set of sz spins takes ceil(sz / n_slots) consecutive rounds
 * (L277: the spins of a set may be updated in any order, or concurrently).  Outputs:
 *   task   [*n_rounds * n_slots][4] (room for 2 N entries): entry e = round * n_slots + slot ->
 *                  byte offsets of the spin's three clause rows (128 t + 64 half_t, in the order
 *                  the kernel accesses them) and, in bits 0-15, the spin index; bit 16 + k is set iff
 *                  this round is the last of the sweep that touches the entry's clause k (the kernels
 *                  for flip tables with w0 > 0 look for ground states there); the whole word =
 *                  0xFFFFFFFF: the slot is idle in that round and its offsets point into scratch line
 *                  N + slot / 2;
 *   place  [N]   : byte offset of clause t's row;
 *   *barrier_mask: bit r set <=> round r is the last round of its set (barrier after it).
 * Guarantees: every spin of a set appears exactly once among the entries of the set's rounds, and
 * slots (2m, 2m+1), which share a shared-memory phase, touch opposite halves in each of their
 * three accesses.  XS_EINVAL if the order needs more than 16 rounds or more than 2 N entries on
 * n_slots slots (n_slots even), or no placement was found.  Any output pointer may be NULL. */
int xs_clause_placement(uint32_t n_spins, uint64_t graph_seed, uint32_t flags, uint32_t set_cap,
                        uint32_t n_slots, uint32_t* task, uint32_t* place, uint32_t* n_rounds,
                        uint32_t* barrier_mask);

/* Launch geometry the library chose for this batch.  No CUDA work. */
int xs_get_layout(const xs_batch* b, xs_layout* out);

/* a-12.  TTS statistics "as the paper defines" (L103-L149) over n_runs runs of one instance
 * with sweep cap t_max: tts[r] = TTS in sweeps or XS_NO_HIT (censored).  t_max = 0 means the runs
 * had no cap; XS_EINVAL if an entry is XS_NO_HIT then (a censored run needs its censoring time).
 * Host only.
 *   out[0] = n (solved runs)                     out[1] = T_tot = sum_solved tts + (n_runs-n) t_max
 *   out[2] = tau_hat = T_tot / n (L139-L147: maximum of the posterior's likelihood; inf if n=0)
 *   out[3..5] = model TTS_50/90/99 = -ln(1-p) tau_hat (L117, L123)
 *   out[6..8] = empirical TTS_50/90/99: the ceil(p n_runs)-th smallest value, censored runs
 *               counting as +inf (L103, L115)
 *   out[9..11] = 16 / 50 / 84 % quantiles of the posterior of tau, inverse-gamma(shape n,
 *               scale T_tot) (L145); for n = 0, out[9] = T_tot / ln 20 (95 % lower bound), rest inf. */
int xs_tts_stats(const uint32_t* tts, uint32_t n_runs, uint64_t t_max, double* out /* [12] */);

/* SURVEY.md 8(f) NEXT-4.  Cavity prediction of the growth rate of the time to solution
 * (Eqs. (3)-(4)): K-spin model on a K-regular random hypergraph at temperature
 * T with a field b that sets the magnetisation m.  With tanh(beta u) = tanh(beta) tanh(beta h)^(K-1),
 * b = h - (K-1) u, m = tanh(beta (u + h)) (Eq. (4)) the free energy along the one-parameter family h is
 *   -beta f = log Z_i + log Z_a - K log Z_ai - beta b m          (Eq. (3); DESIGN.md R-eq3),
 * f_para = -log(2 cosh beta) / beta.  Host only, double precision.
 *   out[0] = beta max_m (f - f_para)  (the barrier; 0.0827249 at K = 3, T_run = -2/ln 0.055, L208)
 *   out[1] = m at the barrier          out[2] = h at the barrier
 *   out[3] = T_sp(K), 1/T_sp = min_x atanh[tanh(x) / tanh((K-1)x)^(K-1)]  (0.980548 for K = 3, L198)
 *   out[4] = beta (f - f_para) of the ferromagnetic state (b = 0, m > 0), out[5] = its m.
 * T >= T_sp: no ferromagnetic solution, out[0..2] and out[4..5] are NaN (out[3] is still set).
 * Returns XS_EINVAL for K < 3 or T <= 0. */
int xs_cavity_barrier(uint32_t K, double T, double* out /* [6] */);

/* Allocation-free ground-state check, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it).  dev_mask [n_instances][n_words] uint64
 * (device, caller-owned): bit b of word w is set iff clone 64 w + b of that instance is in a ground
 * state NOW, i.e. has no unsatisfied interaction, E = -N (the between-launch check of
 * L71) -- the same clones for which xs_energy gives -n_spins.  Asynchronous on cuda_stream.
 * The scratch of the detection kernel (one uint64 per (instance, word)) lives in a static device
 * array inside the library, XS_STATIC_MAX_WORDS words = 512 KiB that every GPU which loads the library
 * holds until exit; the call performs no cudaMalloc / cudaFree and calls no allocating routine.
 * XS_EINVAL if n_instances * n_words > XS_STATIC_MAX_WORDS; XS_ESTATE if the batch's device is not
 * current.  All calls (of all batches, on one GPU) share the array: each clears the part it uses,
 * and calls that OVERLAP on the GPU (different streams without a dependency) race -- serialise them. */
#define XS_STATIC_MAX_WORDS 65536
int xs_solved_mask_static(xs_batch* b, uint64_t* dev_mask /* [inst][W] */, void* cuda_stream);

/* Measurement helpers (no arithmetic of the method).
 * xs_alu_peak: runs a pure-LOP3 micro-kernel (16 independent chains per thread, all SMs) and
 *   returns the measured integer-pipe rate in 32-bit lane-operations per nanosecond for the
 *   whole GPU -- the denominator of the integer-pipe roofline ("P_ALU is
 *   measured").  Synchronises cuda_stream; allocates 4 bytes of device memory for its sink.
 * xs_kernel_launches: kernels launched by this library in this process so far. */
int xs_alu_peak(double* lane_ops_per_ns, double* kernel_ms, void* cuda_stream);
uint64_t xs_kernel_launches(void);

int xs_destroy(xs_batch* b);

const char* xs_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* XS_H_ */
