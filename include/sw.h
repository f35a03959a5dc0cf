/*
 * sw.h -- C ABI of libsw.so: the Swendsen-Wang multi-cluster sweep of a 2D periodic L x L lattice
 * (q-state Potts; q-state clock through Wolff's embedded cluster) on one NVIDIA B200 (sm_100a).
 *
 * Source of the semantics: arXiv 1202.0635 (Komura & Okabe), /root/reference/PAPER.md:
 *   Potts Hamiltonian  H = -J sum_<ij> (delta(S_i,S_j) - 1), periodic            PAPER.md:25-30 eq.(1)
 *   one sweep = bond activation -> cluster labeling -> new state per cluster
 *   proper label of a cluster = its smallest label
 *   clock Hamiltonian  H = -J sum_<ij> S_i . S_j, theta = 2 pi p / q              PAPER.md:132-136 eq.(4)
 *   embedded cluster (Wolff) for the clock model
 *   measurement of energy and magnetisation, M^2 of eq.(3)
 * Everything the paper leaves open (random-number keying, thresholds, clock reflection rule, order
 * of operations) is fixed in DESIGN.md section 3, readings R1..R14.
 *
 * General rules
 *   - J = 1.  Site i = y*L + x (x fastest).  Site i owns the bonds to (x+1 mod L, y) [direction 0]
 *     and (x, y+1 mod L) [direction 1].  Spin values are 0..q-1, one uint8 per site, row-major.
 *   - Every function returning int returns SW_OK (0) or a negative SW_ERR_* code; the two
 *     constructors return a pointer or NULL.  After a failure sw_last_error() describes it.
 *     No exception crosses the boundary.  A context is not thread-safe.
 *   - "host" pointers are ordinary CPU memory owned by the caller; "device" pointers are CUDA
 *     device memory of the current device.  The library never frees caller memory.
 *   - All work of a context is enqueued on its stream.  Functions are synchronous at return
 *     (the stream is synchronised) unless the name ends in _async.
 *   - There is no CPU fallback: if no CUDA device is usable every call fails with SW_ERR_CUDA.
 */
#ifndef SW_H_
#define SW_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct sw_ctx sw_ctx; /* opaque, owned by the library */

enum { SW_POTTS = 0, SW_CLOCK = 1 };
enum { SW_OK = 0, SW_ERR_ARG = -1, SW_ERR_CUDA = -2, SW_ERR_NOMEM = -3, SW_ERR_UNSUPPORTED = -4 };

/* Labeling back-ends (sw_set_algorithm).  Every back-end produces the same spins bit for bit. */
enum {
    SW_ALGO_AUTO = 0,    /* one CTA when L <= 64, else tiled when L allows it, else generic */
    SW_ALGO_GENERIC = 1, /* whole-lattice union-find in global memory; any L >= 2 */
    SW_ALGO_TILED = 2,   /* tile-local union-find in shared memory + boundary merge; needs L % 128 == 0 */
    SW_ALGO_SMALL = 3,   /* one CTA owns the lattice in shared memory and runs all n sweeps of a call in one launch; L <= 128 */
    /* The paper's own labellers, kept as A/B references: whole-lattice label equivalence iterated from
     * the host until a scan changes nothing; any L >= 2.  sw_stats reports their iteration counts. */
    SW_ALGO_HAWICK = 4,  /* Hawick et al.: label + R arrays, scan (atomicMin) / analysis / labeling kernels */
    SW_ALGO_KALENTEV = 5 /* Kalentev et al.: one array, scan / analysis kernels, no atomics */
};

/* Limits of the GPU path: 2 <= L <= 16384 (site index must leave 4 spare bits in an int32 label),
 * 2 <= q <= 16, T finite and > 0, model in {SW_POTTS, SW_CLOCK}.  Violations: NULL / SW_ERR_ARG. */
#define SW_MAX_L 16384
#define SW_MAX_Q 16

/* Bytes of device workspace sw_create_in() needs for this problem (0 if the arguments are invalid). */
size_t sw_workspace_bytes(int L, int q, int model);

/* Create a context; the initial configuration S^0 is drawn from the INIT stream of `seed`
 * (R12) and the sweep index is 0.  sw_create allocates its own device memory and stream.
 * sw_create_in uses caller-owned device memory `d_workspace` (>= sw_workspace_bytes, 256-byte
 * aligned, must outlive the context) and the caller's CUDA stream handle `cuda_stream`
 * (a cudaStream_t cast to void*; NULL = the legacy default stream).  Returns NULL on failure. */
sw_ctx *sw_create(int L, int q, int model, double T, uint64_t seed);
sw_ctx *sw_create_in(int L, int q, int model, double T, uint64_t seed,
                     void *d_workspace, size_t bytes, void *cuda_stream);

/* Destroy a context (NULL is a no-op).  Caller-owned workspace/stream are left untouched. */
void sw_destroy(sw_ctx *ctx);

/* n >= 0 full SW sweeps (steps S0-S4 of DESIGN.md section 1), sweep indices
 * t .. t+n-1 where t = sw_sweep_index().  sw_sweep(a); sw_sweep(b) == sw_sweep(a+b).
 * sw_sweep returns after the work is complete; sw_sweep_async only enqueues it on the stream.
 * Tiled back-end: whole chunks of 16 sweeps are replayed from a CUDA graph (one cudaGraphLaunch per chunk instead of 48
 * kernel launches; the environment variable SW_NO_GRAPH=1, read by sw_create*, turns that off); the result is the same,
 * sw_launch_count counts the replayed kernels, sw_stats out[7] the replays. */
int sw_sweep(sw_ctx *ctx, int n);
int sw_sweep_async(sw_ctx *ctx, int n);
int sw_sync(sw_ctx *ctx);

/* n sweeps with the observables of every configuration recorded ("+ measurement"):
 * row k (q entries) of each HOST output = bond_hist / state_hist of the configuration BEFORE the
 * k-th sweep of this call (R10).  Outputs hold n*q int64 each. */
int sw_sweep_record(sw_ctx *ctx, int n, int64_t *bond_hist_out, int64_t *state_hist_out);

/* Observables of the current configuration, HOST outputs of q int64 each (R11):
 * bond_hist[d] = #{owned bonds with (S_i - S_nbr) mod q == d};  state_hist[k] = #{S_i == k}.
 * Derived doubles: sw_derive_* below. */
int sw_observables(sw_ctx *ctx, int64_t *bond_hist, int64_t *state_hist);

/* NEXT-1 of the scope table: the correlation function of PAPER.md eq.(5) at distance r, as an integer histogram
 * (R15): corr_hist[d] (HOST, q int64) = #{pairs (i, i + r e_x) and (i, i + r e_y), periodic, with
 * (S_i - S_{i+r}) mod q == d}, 2*L*L pairs, of the current configuration; 0 <= r < L.  The caller derives
 * G(r) = (1 / 2N) sum_d corr_hist[d] cos(2 pi d / q) (d ascending) and R = G(L/2) / G(L/4) of eq.(6).
 * sw_sweep_record_corr = sw_sweep_record plus the histograms at the distances r1 and r2 of every configuration
 * ("+ measurement" of the clock model): four HOST outputs of n*q int64. */
int sw_correlation(sw_ctx *ctx, int r, int64_t *corr_hist);
int sw_sweep_record_corr(sw_ctx *ctx, int n, int r1, int r2, int64_t *bond_hist_out, int64_t *state_hist_out,
                         int64_t *corr1_out, int64_t *corr2_out);

/* The doubles the paper plots, derived from the integer histograms above (HOST inputs; plain host arithmetic in a
 * fixed order -- sums run over d or k ascending, left to right, in double; R11, R15).  NaN on invalid
 * arguments (NULL, q outside 2..16, n < 1).
 *   sw_derive_potts_energy  E/J of eq.(1) = 2*L*L - bond_hist[0]
 *   sw_derive_potts_m2      M^2 of eq.(3) = (q sum_k n[k]^2 - N^2) / (q - 1), integer numerator
 *   sw_derive_clock_energy  E/J of eq.(4) = - sum_d bond_hist[d] cos(2 pi d / q)
 *   sw_derive_clock_m       |sum_i S_i| of the planar unit spins, from state_hist
 *   sw_derive_g             G(r) of eq.(5) of one configuration = sum_d corr_hist[d] cos(2 pi d / q) / pairs
 *   sw_derive_moment_ratio  U = <M^4> / <M^2>^2 of eq.(2) over n recorded rows of q state counts
 *   sw_derive_ratio_R       R = <G(L/2)> / <G(L/4)> of eq.(6) over n recorded rows of q pair counts each */
double sw_derive_potts_energy(int L, const int64_t *bond_hist);
double sw_derive_potts_m2(int q, const int64_t *state_hist);
double sw_derive_clock_energy(int q, const int64_t *bond_hist);
double sw_derive_clock_m(int q, const int64_t *state_hist);
double sw_derive_g(int q, const int64_t *corr_hist);
double sw_derive_moment_ratio(int n, int q, const int64_t *state_hist_rows);
double sw_derive_ratio_R(int n, int q, const int64_t *corr_half_rows, const int64_t *corr_quarter_rows);

/* Copy the configuration to / from HOST memory (L*L bytes, row-major, values 0..q-1).
 * sw_set_spins also sets the absolute sweep index (resume / oracle hand-off); values >= q are
 * rejected with SW_ERR_ARG and leave the context unchanged. */
int sw_get_spins(sw_ctx *ctx, uint8_t *host_out);
int sw_set_spins(sw_ctx *ctx, const uint8_t *host_in, uint64_t sweep_index);
uint64_t sw_sweep_index(sw_ctx *ctx); /* 0 for NULL */

/* The integer bond thresholds in use (R6): Potts -> 1 word, clock -> (2q)^2 words,
 * table[ci*2q + cj].  `out` (HOST) may be NULL to query `count` only. */
int sw_get_thresholds(sw_ctx *ctx, uint32_t *out, int *count);

/* Debug exports (HOST outputs).  sw_get_labels: canonical root (minimum site index of the cluster)
 * of every site for the LAST executed sweep, L*L int32 (SW_ERR_ARG before any sweep).
 * sw_debug_bonds: the bonds sweep t = sw_sweep_index() would activate on the current configuration,
 * L*L bytes, bit0 = +x, bit1 = +y; does not advance the state. */
int sw_get_labels(sw_ctx *ctx, int32_t *host_out);
int sw_debug_bonds(sw_ctx *ctx, uint8_t *host_out);

/* Choose the labeling back-end (SW_ALGO_*); SW_ERR_UNSUPPORTED if L does not allow it. */
int sw_set_algorithm(sw_ctx *ctx, int algo);
int sw_get_algorithm(sw_ctx *ctx); /* the back-end actually in use (never SW_ALGO_AUTO) */

/* Labeling work counters accumulated since creation (the analogue of the paper's iteration counts,
 * PAPER.md:75), HOST output of SW_NUM_STATS doubles: out[0] = sweeps counted, out[1] = cross-tile merge attempts,
 * out[2] = tile-local nodes (horizontal runs), out[3] = tile-local union edges, out[4] = pointer hops of the
 * tile-local resolve pass, out[5] = scan passes of the paper's labellers (SW_ALGO_HAWICK / SW_ALGO_KALENTEV, always
 * counted) and out[6] = the sweeps they served (out[5] / out[6] is the iteration count PAPER.md:75 quotes), out[7] = chunks of sweeps replayed from
 * a CUDA graph (always counted), out[8..15] = SM clock cycles the warps of the tile-labeling
 * kernel spent in each of its phases (bonds, setup, run scan, unions, open marking, resolve, output, root decisions;
 * summed over warps).  Counters are only collected after sw_enable_stats(ctx, 1) (they cost atomics and clock reads). */
#define SW_NUM_STATS 16
int sw_enable_stats(sw_ctx *ctx, int on);
int sw_stats(sw_ctx *ctx, double *out);

/* n sweeps with every kernel bracketed by CUDA events on the context's stream (one stream sync per sweep, so
 * this is a measurement mode, not the production path): ms_out[k] (HOST, SW_MAX_KERNELS doubles) receives the
 * summed device time of kernel k over the n sweeps, *n_kernels the number of distinct kernels per sweep of the
 * active back-end; sw_kernel_name(ctx, k) names them (static string, NULL if k is out of range).
 * The configuration advances exactly as with sw_sweep(ctx, n). */
#define SW_MAX_KERNELS 8
int sw_sweep_profile(sw_ctx *ctx, int n, double *ms_out, int *n_kernels);
const char *sw_kernel_name(sw_ctx *ctx, int k);

/* Number of kernel launches this context has enqueued since creation. */
uint64_t sw_launch_count(sw_ctx *ctx);

/* NEXT-2 of the scope table: batches of B independent lattices of the same L, q and model, each with its own
 * temperature T[b] and seed[b] (HOST arrays of B entries) -- the temperature scans of PAPER.md:111-113 (Fig.3),
 * 128-130 (Fig.4), 167-171 (Fig.5), 177-183 (Fig.6) and the small-L rows of Table 1, where one lattice
 * cannot fill a GPU.  Lattice b evolves exactly as a context created with sw_create(L, q, model, T[b], seed[b]) does:
 * same S^0, same spins after every sweep.  L % 128 == 0: the tiles of all lattices in one grid per kernel; other
 * L <= 128: one CTA per lattice, all n sweeps of a call inside one launch.  Other L: NULL / SW_ERR_UNSUPPORTED.
 * HOST buffers: spins B*L*L bytes (lattice-major), histograms B*q int64 each.  The library owns the device memory and
 * the stream of a batch; all calls are synchronous at return. */
#define SW_MAX_BATCH 65536
typedef struct sw_batch sw_batch;
sw_batch *sw_create_batch(int B, int L, int q, int model, const double *T, const uint64_t *seed);
void sw_batch_destroy(sw_batch *batch);
int sw_batch_sweep(sw_batch *batch, int n);
int sw_batch_get_spins(sw_batch *batch, uint8_t *host_out);
int sw_batch_set_spins(sw_batch *batch, const uint8_t *host_in, uint64_t sweep_index);
int sw_batch_observables(sw_batch *batch, int64_t *bond_hist, int64_t *state_hist);
uint64_t sw_batch_sweep_index(sw_batch *batch);

/* NEXT-3 of the scope table: ONE lattice sharded over `nranks` ranks by row stripes (the paper's own outlook, PAPER.md:193;
 * scheme: SURVEY.md 8(e)).  Rank r owns rows [r L / nranks, (r + 1) L / nranks); needs L % nranks == 0 and L % 4 == 0.
 * One sweep is four calls per rank, with two exchanges between them that are the caller's (torch.distributed in
 * paper_1202_0635_b200/stripes.py: NCCL between GPUs, gloo in the CPU test of the host logic):
 *   sw_stripe_first_row    HOST out, L bytes: my first row of spins -- the halo of the previous rank (periodic)
 *   sw_stripe_label        HOST in, L bytes: the first row of the NEXT rank.  Bonds of my sites (Philox keyed on global
 *                          site indices: exactly the bonds of the single-GPU run) and labels inside my stripe
 *   sw_stripe_export_seam  HOST out, L entries each: global index of the local root of every site of my first row, of
 *                          my last row, and whether the +y bond of my last row is active.  All ranks gather these.
 *   sw_seam_solve          pure host code (no device needed), identical on every rank: first / last / seam are the
 *                          gathered [nranks][L] arrays; union-find by minimum index over the seam pairs; out: the local
 *                          roots whose canonical root differs from themselves, from[k] -> to[k], k < *n_map <= 2 nranks L
 *   sw_stripe_finish       HOST in: that map.  Decisions keyed on the global canonical root, spin update; sweep index + 1
 * The spins after every sweep equal those of the single-GPU run bit for bit.  sw_stripe_get_labels: canonical roots of
 * the last finished sweep (rows * L int32).  NULL / SW_ERR_* as everywhere. */
typedef struct sw_stripe sw_stripe;
sw_stripe *sw_stripe_create(int L, int q, int model, double T, uint64_t seed, int rank, int nranks);
void sw_stripe_destroy(sw_stripe *stripe);
int sw_stripe_first_row(sw_stripe *stripe, uint8_t *host_out);
int sw_stripe_label(sw_stripe *stripe, const uint8_t *halo_row_host);
int sw_stripe_export_seam(sw_stripe *stripe, int32_t *first_row_labels, int32_t *last_row_labels, uint8_t *seam_bonds);
int sw_seam_solve(int nranks, int L, const int32_t *first, const int32_t *last, const uint8_t *seam, int32_t *from, int32_t *to, int *n_map);
int sw_stripe_finish(sw_stripe *stripe, int n_map, const int32_t *from, const int32_t *to);
int sw_stripe_get_spins(sw_stripe *stripe, uint8_t *host_out);
int sw_stripe_get_labels(sw_stripe *stripe, int32_t *host_out);
int sw_stripe_set_spins(sw_stripe *stripe, const uint8_t *host_in, uint64_t sweep_index);
uint64_t sw_stripe_sweep_index(sw_stripe *stripe);

/* Instruction-issue probes (measurement infrastructure for the "alu" roofline of DESIGN.md section 6; the sweep never
 * uses them).  Probe `probe` (0 .. until sw_microbench_name returns NULL) runs `warps_per_smsp` (1..16) warps on every
 * SM sub-partition of the current device, each executing `iters` loop iterations of 8 independent dependency chains of
 * one SASS instruction (or a fixed mix, or whole Philox4x32-10 calls).  out (HOST, 4 doubles): [0] = units retired per
 * SM clock cycle per sub-partition (a unit = one warp-instruction, one pair, or one Philox call, as the name says),
 * [1] = SM cycles of the slowest CTA, [2] = of the fastest, [3] = units per sub-partition. */
int sw_microbench(int probe, int warps_per_smsp, int iters, double *out);
const char *sw_microbench_name(int probe);

/* Device self-test of the kernels' carry-flag threshold compares ([word >= threshold] shifted in through add.cc / sub.cc
 * + addc) against the plain comparison over edge values on the current device: SW_OK, or SW_ERR_UNSUPPORTED if the
 * toolchain's carry convention differs from the one the kernels were written for (every clock bond would flip). */
int sw_selftest(void);

/* One sweep WITHOUT any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): no context, no workspace argument.  The scratch of the sweep (clock threshold
 * table, bonds S1, union-find parents S2: 4096 + 5 * SW_NOALLOC_MAX_L^2 bytes = 5 MiB + 4 KiB) is a file-scope
 * `static __device__` array of libsw.so; every GPU that loads the library holds it until the process exits.
 *   d_spins_out = the configuration sweep `sweep_index` (S1..S4 of the generic back-end) makes of
 *   d_spins_in, bit for bit what sw_create(L, q, model, T, seed); sw_set_spins(in, sweep_index); sw_sweep(1);
 *   sw_get_spins(out) gives with any back-end.
 * d_spins_in, d_spins_out: DEVICE memory of the current device, L*L bytes each, row-major, owned by the caller;
 * they may be the same buffer but must not overlap partially.  Values >= q are NOT checked (the result is then
 * unspecified, but no access leaves the scratch or the two buffers).  cuda_stream: a cudaStream_t of the current
 * device, or NULL for the default stream.  The call is ASYNCHRONOUS: it enqueues one small copy (clock model only, the
 * threshold table, from host stack memory) and 5 kernels on the stream and returns; synchronise the stream before
 * reading d_spins_out.  It calls no cudaMalloc, cudaFree or allocating library routine; the address of the scratch is
 * taken once per device with cudaGetSymbolAddress.
 * Limits: 2 <= L <= SW_NOALLOC_MAX_L (larger L: SW_ERR_UNSUPPORTED, nothing enqueued), q, T, model as for sw_create,
 * sweep_index <= 2^32-1.
 * Every call on a device shares the one scratch array, which keeps the previous call's contents: each call rewrites
 * all of it that it reads (nothing has to start at zero), and calls are ordered only by their streams -- two calls
 * that overlap on the GPU (different streams, or different host threads on different streams) RACE on the scratch and
 * give garbage.  Calls on the same stream, or otherwise ordered, are safe. */
#define SW_NOALLOC_MAX_L 1024
int sw_sweep_noalloc(int L, int q, int model, double T, uint64_t seed, uint64_t sweep_index,
                     const uint8_t *d_spins_in, uint8_t *d_spins_out, void *cuda_stream);

/* Thread-local description of the last failure in this thread ("" if none). */
const char *sw_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SW_H_ */
