/*
 * ff.h -- C ABI of the B200-native Barnes-Hut dipole field + force library.
 *
 * Hot path of arxiv 1212.2934 ("Large-scale Ferrofluid Simulations on Graphics
 * Processing Units"): for N magnetic particles with positions rho_k and moment
 * directions u_k (reduced units) compute, per
 * particle,
 *     h_k = sum_{j != k} [3 rho_kj (u_j.rho_kj) - u_j rho_kj^2] / rho_kj^5        (Eq. 10-11, no h_ext)
 *     f_k = sum_{j != k} { 3 [rho_kj (u_j.u_k) + u_k (u_j.rho_kj) + u_j (u_k.rho_kj)] / rho_kj^5
 *                          - 15 rho_kj (u_k.rho_kj)(u_j.rho_kj) / rho_kj^7 }       (Eq. 12)
 * with rho_kj = rho_k - rho_j, either exactly (all pairs) or with
 * the Barnes-Hut octree approximation: a cell's particles are
 * replaced by one pseudo-particle with u' = sum u_i at rho' = (sum rho_i)/N'
 * (Eq. 14) when the cell is far enough.
 *
 * Conventions
 *  - All particle arrays are fp32, shape [N][3], C-contiguous, in CALLER order.
 *    "device" = pointer to CUDA device memory of the current device,
 *    "host"   = pointer to host memory (pinned memory makes the copies async).
 *  - The caller owns every array and the workspace.  After ff_create the
 *    library allocates no device memory and, inside build/eval/step, reads no
 *    device data back to the host.
 *  - Calls enqueue work on the context's stream and return; only the ff_get_*
 *    and *_host functions synchronise that stream.
 *  - Return value: FF_OK (0) or a negative ff_status.  No exceptions cross the
 *    ABI.  One context per host thread; a context is bound to the device that
 *    was current at ff_create: every call makes that device current while it runs
 *    and restores the caller's device before it returns.
 *  - Undefined input (documented, not checked): non-finite values; two
 *    distinct particles at the same position (r = 0 gives inf/NaN exactly as
 *    in Eq. 11; the paper prevents it with the Lennard-Jones core);
 *    ff_eval_bh called with a `pos` array whose CONTENT changed since ff_build_tree (the pointer is checked).
 *  - Units: the path is unit free (h ~ L^-3, f ~ L^-4).
 */
#ifndef FF_H
#define FF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ff_ctx ff_ctx;   /* opaque */

typedef enum ff_status {
    FF_OK = 0,
    FF_ERR_INVALID_ARG = -1,    /* NULL pointer, N <= 0, N > FF_MAX_N, theta < 0 or NaN, unknown option */
    FF_ERR_WORKSPACE = -2,      /* workspace NULL, too small or not 256-byte aligned */
    FF_ERR_NO_TREE = -3,        /* ff_eval_bh / ff_get_tree before ff_build_tree */
    FF_ERR_CAPACITY = -4,       /* internal pool overflow (cannot happen with ff_workspace_bytes' sizing; kept for the ABI).
                                   Detected on the device, reported by the next ff_get_tree / ff_get_timings / ff_get_counters */
    FF_ERR_CUDA = -5,           /* CUDA runtime / launch failure; text via ff_last_error */
    FF_ERR_CHECK = -6,          /* checked build only (library compiled with -DFF_CHECKED): a device-side index or bound
                                   check failed; reported like FF_ERR_CAPACITY, the failing source line is in
                                   ff_last_error after the reporting call */
    FF_ERR_TOO_LARGE = -7       /* ff_eval_direct_static only: n > FF_STATIC_MAX_N (its scratch array has a fixed size) */
} ff_status;

#define FF_MAX_N (1ll << 28)    /* particle slots must fit the 30-bit stack entries of the walk */
#define FF_MAX_LEVEL 10         /* 30-bit Morton key = 10 octant digits */

/* ff_set_option keys */
enum {
    FF_OPT_THETA = 1,     /* opening parameter theta >= 0 ("large enough": s/d < theta) */
    FF_OPT_NLEAF = 2,     /* leaf capacity N_leaf >= 1; 1 = the paper's tree. Invalidates the tree. */
    FF_OPT_COUNTERS = 3,  /* != 0: the walk also counts interactions (slower); read with ff_get_counters */
    FF_OPT_TIMING = 4,    /* != 0: record CUDA events around each phase; read with ff_get_timings */
    FF_OPT_CELL_ORDER = 6, /* 0 (default): a cell acts as the paper's pseudo-particle, Eq. 14.  1: plus the
                             first-order term of the expansion of Eq. 11-12 about the cell centre, with the cell tensor
                             D = sum_i (rho_i - rho') (x) u_i (not in the paper).
                             Same interaction lists; W = 32 only */
    FF_OPT_GROUP = 5      /* targets per walk group W (reading Q2): 32 (default) or 64, one warp per group with
                             two targets per lane; any other value is FF_ERR_INVALID_ARG (the oracle takes any W) */
};

/* phases reported by ff_get_timings, in launch order */
enum {
    FF_PH_BBOX_KEYS = 0,  /* a1 bounding box + a2 Morton keys        */
    FF_PH_SORT = 1,       /* a3 radix sort of (key, index) + gather        */
    FF_PH_BUILD = 2,      /* a4 octree from the sorted keys   */
    FF_PH_MOMENTS = 3,    /* a5 cell pseudo-particles, Eq. 14*/
    FF_PH_WALK = 4,       /* a6 tree walk + a7 scatter to caller order   */
    FF_PH_DIRECT = 5,     /* a8 tiled all-pairs    */
    FF_PH_STEP = 6,       /* integration update (ff_step)        */
    FF_N_PHASES = 7
};

/*
 * Bytes of device workspace ff_create needs for up to N particles: key/index
 * double buffers, sorted float4 copies, the worst-case node pool (an octree
 * over 30-bit keys whose internal cells hold >= 2 particles has at most 5N
 * internal cells), scan and sort scratch.  Returns 0 if N is out of range.
 */
size_t ff_workspace_bytes(int64_t N);

/*
 * Create a context for up to N particles with opening parameter theta.
 * workspace: device pointer, 256-byte aligned, >= ff_workspace_bytes(N) bytes,
 * owned by the caller and kept alive until ff_destroy.  The context uses the
 * legacy default stream until ff_set_stream is called.
 */
int ff_create(ff_ctx** out, int64_t N, float theta, void* workspace, size_t workspace_bytes);
int ff_destroy(ff_ctx* ctx);

/* cuda_stream: a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream. */
int ff_set_stream(ff_ctx* ctx, void* cuda_stream);
int ff_set_option(ff_ctx* ctx, int key, double value);

/*
 * a1-a4: bounding box -> root cube -> 30-bit Morton keys ->
 * stable radix sort -> sorted float4 positions -> octree.  pos: device,
 * [n][3] fp32, n <= N of ff_create (n = number of particles of this call).
 * Tree definition (readings O3): root cube anchored at the min
 * corner with side S = largest extent (S = 1 if all points coincide); grid
 * coordinate q_a = min(1023, floor(fl(fl(pos_a - lo_a) * fl(1024 / S)))) in
 * fp32 round-to-nearest; key bit 3b+2/3b+1/3b = bit b of q_x/q_y/q_z; stable
 * order (ties keep caller order); the level-l cell with prefix P is the range
 * of sorted particles whose top 3l key bits equal P; a cell with more than
 * N_leaf particles and l < 10 is internal.
 */
int ff_build_tree(ff_ctx* ctx, const float* pos, int64_t n);

/*
 * a5-a7: cell moments (Eq. 14) -> tree walk -> results in caller order.
 * pos must be the array the tree was built from (another pointer is FF_ERR_INVALID_ARG); mom: device [n][3] fp32
 * (need not be unit length: Eq. 11-12 are bilinear in the moments).
 * H_out / F_out: device [n][3] fp32, either may be NULL to skip it.
 * H_out = sum_{j != k} h_kj only (no external field); F_out = f_k of Eq. 12,
 * no prefactor.  Opening rule (reading O5): targets are walked in
 * groups of W = 32 (FF_OPT_GROUP: or 64) consecutive sorted particles (one warp); a leaf's particles
 * are summed directly (self skipped by index); an internal cell is opened if
 * its range holds a member of the group, else accepted for the whole group
 * iff every member k satisfies, in fp32 and exactly this order,
 *   d2 = fma(dz,dz, fma(dy,dy, fl(dx*dx))),  fl(s_l*s_l) < fl(fl(theta*theta) * d2)
 * with (dx,dy,dz) = fl(p_k - rho') and s_l = S 2^-l; else opened.
 */
int ff_eval_bh(ff_ctx* ctx, const float* pos, const float* mom, float* H_out, float* F_out);

/*
 * The same for a slice of the targets: only the walk groups [group_begin, group_end) of the SORTED order are
 * evaluated (group g = sorted slots W g .. W g + W - 1; group_end < 0 means "to the last group"), and only the
 * rows of H_out / F_out that belong to those targets (caller order, scattered) are written.  The cell moments are
 * computed for the whole tree.  This is the unit of the target sharding of SURVEY.md 8(e): every GPU holds all
 * sources and the whole tree and evaluates a Morton-contiguous slice of the targets; no halo, no reduction.
 */
int ff_eval_bh_range(ff_ctx* ctx, const float* pos, const float* mom, float* H_out, float* F_out,
                     int64_t group_begin, int64_t group_end);

/*
 * a8: exact all-pairs sum (Algorithm 1), self excluded by
 * index (line 5).  Needs no tree.  Arguments as ff_eval_bh, n given.
 */
int ff_eval_direct(ff_ctx* ctx, const float* pos, const float* mom, int64_t n, float* H_out, float* F_out);

/*
 * The same all-pairs sum (a8, Algorithm 1) for callers that must not allocate device memory.
 *
 * Who that is: code that runs after a framework's memory pool has claimed the whole GPU, so that a cudaMalloc of
 * its own fails or fights the pool; code inside a latency-critical loop, where cudaMalloc / cudaFree stall the
 * whole device; and plug-ins that are handed fixed input and output buffers and nothing they could use as the
 * workspace ff_create asks for.  For n of a few thousand the all-pairs kernel splits the sources over the grid and
 * needs somewhere to keep one fp64 partial sum per (split, target) until they are added up; ff_eval_direct keeps
 * them in the caller's workspace, this call keeps them in an array that is compiled into the library.
 *
 *  - No context, no workspace; the call makes no cudaMalloc, cudaFree or other allocating call.  The array is
 *    3 MiB of device memory that EVERY GPU on which this library gets loaded holds until the process exits,
 *    whether or not this function is ever called there.
 *  - n <= FF_STATIC_MAX_N (what the array can hold); a larger n returns FF_ERR_TOO_LARGE and launches nothing.
 *  - pos, mom: device [n][3] fp32; H_out, F_out: device [n][3] fp32, one of them may be NULL.  All arrays and
 *    cuda_stream (a cudaStream_t; NULL = default stream) must belong to the CURRENT device; the work is
 *    enqueued on that stream and the call returns without synchronising.
 *  - The first call on each device looks up the array's device address (cudaGetSymbolAddress, which may also load
 *    the library's kernels onto that device).  Make that first call outside any stream capture.
 *  - All calls share the one array, and it keeps whatever the last call left in it.  That is harmless for calls
 *    that follow one another on the GPU (every record a call reads it has written itself first; nothing relies on
 *    zeros), but two calls whose kernels can run at the same time on one GPU -- different streams, no event
 *    between them -- overwrite each other's partial sums and return garbage.  Order them yourself.
 *  - Results: the same arithmetic as ff_eval_direct (the same kernels); they agree to rounding order, and bit for
 *    bit whenever both pick the same number of source splits.
 * Returns FF_OK or a negative ff_status; ff_static_last_error() has the text of this thread's last failure.
 */
#define FF_STATIC_MAX_N 32768
int ff_eval_direct_static(const float* pos, const float* mom, int64_t n, float* H_out, float* F_out,
                          void* cuda_stream);
/* Text of the calling thread's last ff_eval_direct_static failure ("" after a success). */
const char* ff_static_last_error(void);

/*
 * End-to-end convenience calls with HOST buffers: copy pos/mom to the device
 * (staging space inside the workspace), run ff_build_tree + ff_eval_bh (or
 * ff_eval_direct), copy H/F back, synchronise.  H_host / F_host may be NULL.
 */
int ff_eval_bh_host(ff_ctx* ctx, const float* pos_host, const float* mom_host, int64_t n,
                    float* H_host, float* F_host);
/*
 * The same without the final synchronise: enqueues upload, ff_build_tree + ff_eval_bh and download and returns.
 * Uploads, compute and downloads use three streams and two sets of staging buffers, so in a sequence of calls
 * the copies of one call overlap the compute of its neighbours.  The host buffers must be page-locked for the
 * copies to be asynchronous and must not be touched (inputs: not modified; outputs: not read) before
 * ff_host_sync returns.  At most two calls are in flight on the device; a third waits on the GPU, not on the host.
 */
int ff_eval_bh_host_async(ff_ctx* ctx, const float* pos_host, const float* mom_host, int64_t n,
                          float* H_host, float* F_host);
/* Block until every *_host call issued on this context has delivered its results. */
int ff_host_sync(ff_ctx* ctx);
int ff_eval_direct_host(ff_ctx* ctx, const float* pos_host, const float* mom_host, int64_t n,
                        float* H_host, float* F_host);

/*
 * One Euler-Maruyama step (dtau) of the reduced equations of
 * motion Eq. 7-9 in the vector form of DESIGN.md (reading
 * Q12): rebuilds the tree from pos, evaluates h and f^dip with Barnes-Hut,
 * adds the external field (Eq. 10) and the Lennard-Jones force (Eq. 13,
 * PAPER.md:74, pairs within lj_cutoff), then updates in place
 *   pos    += dtau vel
 *   vel    += dtau (f^dip + f^sr - gamma_d vel) + noise_d sqrt(dtau) xi_d
 *   angvel += dtau 5/2 (u x h - gamma_r angvel) + noise_r sqrt(dtau) xi_r
 *   mom     = normalise(mom + dtau angvel x mom)
 * (explicit: every right-hand side uses the values at the start of the step)
 * All arrays device [n][3] fp32.  noise_* = 0 gives the deterministic step
 * used by the parity tests; otherwise xi are unit Gaussians from a
 * counter-based generator keyed by (seed, step_index, particle, component).
 * Streams: the call is ordered on the context's stream like every other call (work enqueued on that stream after
 * ff_step returns sees the updated state).  Internally the Lennard-Jones pass, which needs the tree but not the
 * fields, runs on a second stream of the context beside the tree walk (same priority as the caller's stream on
 * current GPUs: how far the two overlap depends on submission timing); the update waits for both.  All parameter
 * checks run before anything is enqueued: a call that returns FF_ERR_INVALID_ARG has launched nothing.
 */
typedef struct ff_step_params {
    float dtau;          /* time step (paper: 0.001) */
    float gamma_d;       /* translational drag Gamma_d */
    float gamma_r;       /* rotational drag Gamma_r */
    float h_ext[3];      /* reduced external field (Eq. 10) */
    float lj_epsilon;    /* epsilon of Eq. 13; 0 disables the short-range force */
    float lj_sigma;      /* sigma of Eq. 13 in the unit of pos (force vanishes at rho = sigma) */
    float lj_cutoff;     /* pairs with rho < lj_cutoff contribute */
    float noise_d;       /* amplitude multiplying sqrt(dtau) xi in the velocity update (0 = off) */
    float noise_r;       /* same for the angular velocity */
    uint64_t seed;
    /* container walls (reading Q20): the six planes of the box [wall_lo, wall_hi]
     * act on a particle at distance d < lj_cutoff with 24 wall_epsilon / d [ (wall_sigma/d)^12 - (wall_sigma/d)^6 ]
     * along the inward normal.  wall_epsilon = 0 disables the walls; particles must start inside the box. */
    float wall_lo[3];
    float wall_hi[3];
    float wall_epsilon;
    float wall_sigma;    /* centre-to-wall distance at which the wall force vanishes */
    int32_t all_pairs;   /* != 0: h^dip, f^dip and f^sr by the exact all-pairs sum (the paper's Algorithm 1; no tree).
                            The faster choice below N ~ 10^4 */
    int32_t reserved;    /* 0 */
} ff_step_params;

int ff_step(ff_ctx* ctx, float* pos, float* vel, float* mom, float* angvel, int64_t n,
            const ff_step_params* p, uint64_t step_index);

/*
 * Introspection for tests and measurement.  Pointers are DEVICE pointers into
 * the workspace, valid until the next ff_build_tree / ff_step / ff_destroy.
 * Synchronises the stream.  Internal cells are numbered in pre-order, i.e.
 * sorted by (first, level).  child[8*i + j], j = 0..7, are the sub-cells of cell i COMPACTED: the non-empty ones
 * first, in octant order (0..7 = 4x + 2y + z), then FF_CHILD_EMPTY for the rest:
 *   FF_CHILD_EMPTY                         no further sub-cell
 *   v >= 0                                 internal cell v
 *   (v & FF_CHILD_LEAF1) == FF_CHILD_LEAF1 and not MULTI: single-particle leaf, slot = v & FF_CHILD_SLOT
 *   FF_CHILD_MULTI set                     leaf with leaf_count[slot] > 1 particles starting at slot
 */
#define FF_CHILD_EMPTY  ((int32_t)-1)
#define FF_CHILD_LEAF1  0x80000000u
#define FF_CHILD_MULTI  0x40000000u
#define FF_CHILD_SLOT   0x3FFFFFFFu

typedef struct ff_tree_view {
    int64_t n;                 /* particles in the tree */
    int64_t n_cells;           /* internal cells (0 when n <= N_leaf: the root is a leaf) */
    int32_t nleaf;
    float lo[3];               /* root cube origin */
    float S;                   /* root cube side */
    const uint32_t* key;       /* [n] sorted Morton keys */
    const uint32_t* perm;      /* [n] perm[s] = caller index of sorted slot s */
    const float* pos_sorted;   /* [n][4] x,y,z,unused */
    const float* mom_sorted;   /* [n][4] valid after ff_eval_bh */
    const int32_t* cell_first; /* [n_cells] first sorted slot */
    const int32_t* cell_end;   /* [n_cells] one past the last slot */
    const int32_t* cell_level; /* [n_cells] */
    const int32_t* child;      /* [n_cells][8] */
    const int32_t* leaf_count; /* [n] defined at the first slot of multi-particle leaves */
    const float* cell_centre;  /* [n_cells][4] rho'.xyz (fp32), fl(s_l^2); valid after ff_eval_bh */
    const float* cell_moment;  /* [n_cells][4] u'.xyz (fp32), N' as float; valid after ff_eval_bh */
    const float* cell_quad;    /* [n_cells][8] symmetric part of the cell tensor D, xx yy zz xy xz yz 0 0 (fp32).  Non-NULL only
                                  if the last ff_eval_bh on this tree ran with FF_OPT_CELL_ORDER = 1 (NULL before any
                                  evaluation and after an order-0 one: the array would hold stale tensors) */
} ff_tree_view;

int ff_get_tree(ff_ctx* ctx, ff_tree_view* out);

/* CUDA-event milliseconds per phase of the calls since the last ff_get_timings (needs FF_OPT_TIMING).  After ff_step
 * with a Lennard-Jones force, FF_PH_WALK and FF_PH_STEP include whatever of the concurrent Lennard-Jones kernels ran
 * inside their event brackets (second stream). */
int ff_get_timings(ff_ctx* ctx, float ms[FF_N_PHASES]);

/*
 * Interaction counts of the last ff_eval_bh (needs FF_OPT_COUNTERS):
 * n_cell = accepted-cell terms summed over targets, n_particle = direct
 * particle terms summed over targets (self excluded), n_mac_tests = opening
 * tests (group, internal cell not holding a member) evaluated.
 */
int ff_get_counters(ff_ctx* ctx, uint64_t* n_cell, uint64_t* n_particle, uint64_t* n_mac_tests);

/*
 * How many of the n_mac_tests of the last ff_eval_bh the walk's cheap pre-filter (group bounding box +
 * four probe members) could not decide and passed on to the full 32-member test
 * (needs FF_OPT_COUNTERS).  A measurement aid: the decisions themselves are unaffected.
 */
int ff_get_prefilter_count(ff_ctx* ctx, uint64_t* n_parked);

/* Number of kernel launches issued by this context since creation (for bench accounting). */
int ff_get_launch_count(ff_ctx* ctx, uint64_t* launches);

/*
 * FP32 FMA-pipe microbenchmark: runs `iters` dependent-chain FFMA per thread
 * with 8 independent chains on a full grid and returns achieved TFLOP/s
 * (2 flop per FMA) measured with CUDA events.  Used by bench.py as the
 * measured ALU peak next to the nominal SMs x 128 x 2 x clock.
 */
int ff_measure_fp32_peak(ff_ctx* ctx, int iters, double* tflops);

/*
 * The other FP32-pipe probes (same calling convention, result in TFLOP/s with an FMA counted as 2 flop):
 * what the ALU roofline of ff_k_walk / ff_k_direct is measured against.
 *   FF_PROBE_FFMA          the scalar FFMA chains of ff_measure_fp32_peak
 *   FF_PROBE_FFMA2_PAIRS   packed FFMA2 with three distinct register-pair operands
 *   FF_PROBE_FFMA2_REUSE   packed FFMA2 with one operand shared by consecutive instructions (operand reuse cache)
 *   FF_PROBE_FFMA2_SCALAR  packed FFMA2 with one scalar operand in the broadcast form (how the sources enter Eq. 11-12)
 *   FF_PROBE_EVAL          the evaluation loop of the walk alone: 36 packed FP32 instructions (force as a tensor) + 2 MUFU.RSQ per source
 *                          and pair of targets on shared-memory records, 60 flop per interaction -- the ceiling of the
 *                          walk and of the direct kernel AS ENCODED in packed FP32
 *   FF_PROBE_EVAL_SCALAR   the same 36 operations per target on scalars (72 FFMA / FMUL per source and pair of targets)
 *   FF_PROBE_EVAL_HYBRID   packed except for the twelve FFMA2 with three different register-pair operands, which run as
 *                          24 scalar FFMA -- together with _SCALAR the evidence for whether the packed form's operand
 *                          bandwidth or the arithmetic bounds that loop
 */
enum {
    FF_PROBE_FFMA = 0,
    FF_PROBE_FFMA2_PAIRS = 1,
    FF_PROBE_FFMA2_REUSE = 2,
    FF_PROBE_FFMA2_SCALAR = 3,
    FF_PROBE_EVAL = 4,
    FF_PROBE_EVAL_SCALAR = 5,
    FF_PROBE_EVAL_HYBRID = 6
};
int ff_measure_probe(ff_ctx* ctx, int kind, int iters, double* tflops);

const char* ff_error_string(int code);
/* Text of the last CUDA error seen by this context ("" if none). */
const char* ff_last_error(ff_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* FF_H */
