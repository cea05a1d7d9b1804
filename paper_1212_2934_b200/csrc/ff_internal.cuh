// ff_internal.cuh -- context layout and launch helpers shared by the .cu files of libff.
// Nothing here is visible through include/ff.h.  sm_100a only.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/ff.h"

#define FF_WARP 32
#define FF_FULL 0xffffffffu

// ---- radix sort geometry (ff_sort.cu) --------------------------------------
#define FF_SORT_THREADS 256
#ifndef FF_SORT_ROUNDS
#define FF_SORT_ROUNDS 8                                   // keys per thread
#endif
#define FF_SORT_TILE (FF_SORT_THREADS * FF_SORT_ROUNDS)    // keys per block
#define FF_RADIX_BITS 8
#define FF_RADIX 256
#define FF_SORT_PASSES 4

// ---- scan geometry (ff_build.cu) --------------------------------------------
#define FF_SCAN_THREADS 256
#define FF_SCAN_ITEMS 8
#define FF_SCAN_TILE (FF_SCAN_THREADS * FF_SCAN_ITEMS)
#define FF_BUILD_MAX_BLOCKS 4096     // grid limit of ff_k_build (its per-block counts live in scan_blk)

// ---- walk geometry (ff_walk.cu) ---------------------------------------------
#ifndef FF_WALK_WARPS
#define FF_WALK_WARPS 4            // warps (= target groups) per block
#endif
#ifndef FF_WALK_MINB
#define FF_WALK_MINB 5             // min resident blocks per SM asked of ptxas (caps registers at 96; 5 x 4 warps per SM)
#endif
#ifndef FF_WALK_MINB_QUAD
#define FF_WALK_MINB_QUAD 4        // the same for the order-1 walk: 119 registers at 4; 5 (95 registers, no spills) measured slower, DESIGN.md 8b
#endif
#define FF_WALK_STACK 1024         // traversal stack entries per warp
#ifndef FF_WALK_BATCH
#define FF_WALK_BATCH 64           // ring entries evaluated in one go
#endif
#define FF_WALK_PEND (2 * FF_WALK_BATCH)   // pending interaction ring per warp (two batches)
#ifndef FF_WALK_PROBE_PAIRS
#define FF_WALK_PROBE_PAIRS 2      // probe members (x2) of the opening pre-filter: the members at the x and y extremes
#endif                             // of the group's box
#define FF_WALK_AMB_ROOM 256       // stack room an ambiguous-queue round may need (32 cells x 8 children)

// ---- direct geometry (ff_direct.cu) -------------------------------------------
#define FF_DIRECT_THREADS 256
#define FF_DIRECT_SPLIT_ELEMS (1 << 19)   // max targets*splits whose partial sums fit the scratch

// Small block of device-resident scalars: written and read by kernels only, so
// that build/eval never needs a host read (SURVEY.md 8(b) "no host round-trip").
struct ff_globals {
    uint32_t bbox_ord[8];     // ordered-uint encoding of min xyz [0..2] and max xyz [4..6]
    float lo[3];              // root cube origin
    float S;                  // root cube side
    float inv;                // fl(1024 / S)
    int32_t n_cells;          // internal cells of the current tree
    int32_t error;            // sticky device-side error flag (FF_ERR_*)
    int32_t check_line;       // FF_CHECKED: source line of the first failed device-side check
    int32_t max_level;        // deepest level holding an internal cell
    int32_t level_count[FF_MAX_LEVEL];      // internal cells per level (ff_k_build)
    int32_t level_cursor[FF_MAX_LEVEL];     // fill cursors of the level lists
    int32_t level_start[FF_MAX_LEVEL + 1];  // cell_list[level_start[l] .. level_start[l+1]) = the cells of level l
    int32_t walk_next;        // next target group of the persistent walk (zeroed by the level-0 moment launch)
    unsigned long long counters[4];   // n_cell, n_particle, n_mac, n_parked (FF_OPT_COUNTERS)
    int32_t sort_ticket[FF_SORT_PASSES];              // next tile of each sort pass
    uint32_t digit_hist[FF_SORT_PASSES][FF_RADIX];    // global digit histograms of the four passes (ff_k_keys)
};

struct ff_ctx {
    int64_t N;                // capacity
    int64_t n;                // particles of the current tree / call
    int64_t cell_cap;         // capacity of the cell pool
    float theta;
    int nleaf;
    int count_enabled;
    int timing_enabled;
    int tree_built;
    int globals_clean;        // the device-side build state (bbox, sort tickets, digit histograms) is reset: set by a
                              // completed ff_build_tree (ff_k_build resets it for the next one), cleared while one runs
    const float* tree_pos;    // the pos array the current tree was built from (ff_eval_bh checks it is given the same one)
    int moments_valid;
    int moments_order;        // the FF_OPT_CELL_ORDER the current cell data was computed with (cell_quad is defined iff 1)
    int device;
    int num_sms;
    int group;                // targets per walk group W: 32 or 64 (FF_OPT_GROUP)
    int order;                // 0 = the paper's cell (Eq. 14), 1 = plus the first-order cell term (FF_OPT_CELL_ORDER)
    int occ_walk[12], occ_build, occ_moments[2];   // resident blocks per SM of the persistent / cooperative kernels (0 = not queried yet)
    cudaStream_t stream;
    // pipelined *_host calls: uploads on in_stream, compute on `stream`, downloads on out_stream, staging
    // buffers and events double-buffered by call parity (ff_api.cu)
    cudaStream_t in_stream, out_stream;
    cudaEvent_t ev_pos[2], ev_in[2], ev_done[2], ev_out[2];
    // ff_step: the Lennard-Jones pass needs the tree only, not the walk's results; it runs on a second
    // stream beside the walk and can fill the SMs the draining walk leaves idle (ff_api.cu)
    cudaStream_t lj_stream;
    cudaEvent_t ev_tree, ev_lj;
    uint64_t host_seq;                // *_host calls issued so far
    uint64_t launches;
    char last_error[256];

    // workspace carve-up (device pointers)
    char* ws; size_t ws_bytes;
    ff_globals* g;
    uint32_t *key[2], *idx[2];        // ping-pong buffers of the sort; result in [0]
    float4 *pos_s, *mom_s;            // sorted particles
    int32_t* leaf_count;              // [N]
    int32_t* cell_base;               // [N] exclusive scan of cells starting at each slot
    uint32_t* scan_blk;               // block sums of the scan
    uint32_t* sort_status;            // [FF_SORT_PASSES][n_tiles][FF_RADIX] look-back status words
    int32_t *cell_first, *cell_end, *cell_level;
    int4* cell_info;                  // [cap] first, end, number of children, level: what the walk reads per cell
    int32_t* cell_list;               // [cap] cell ids grouped by level
    int32_t* cell_child;              // [cap][8]
    float4 *cell_centre, *cell_moment;
    double* cell_sums;                // [cap][8] fp64 sums in the fixed order: u.xyz, p.xyz, 2 pad (64-byte records)
    double* cell_sums2;               // [cap][8] FF_OPT_CELL_ORDER = 1: sums of the symmetrised rho (x) u, xx yy zz xy xz yz, 2 pad
    float4* cell_quad;                // [cap][2] the cell tensor D: (xx, yy, zz, xy) (xz, yz, 0, 0)
    double* direct_part;              // partial sums of the split direct kernel
    float *stage_pos2[2], *stage_mom2[2], *stage_H2[2], *stage_F2[2];   // device staging of the *_host calls
    float *stage_H, *stage_F;         // = stage_H2[0], stage_F2[0]: the fields of ff_step
    float* step_fsr;                  // [N][3] short-range force (ff_step)

    cudaEvent_t ev[FF_N_PHASES][2];
    int ev_valid[FF_N_PHASES];
};

// Makes the context's device current for the duration of an ABI call and restores the caller's afterwards (a context
// is bound to the device that was current at ff_create; the caller may have switched since).
struct ff_device_guard {
    int prev = -1, dev = -1;
    explicit ff_device_guard(const ff_ctx* c)
    {
        if (!c) return;
        dev = c->device;
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) cudaSetDevice(dev); else prev = -1;
    }
    ~ff_device_guard() { if (prev >= 0) cudaSetDevice(prev); }
};

// ---- error plumbing ------------------------------------------------------------
static inline int ff_cuda_fail(ff_ctx* c, cudaError_t e, const char* what)
{
    if (c) snprintf(c->last_error, sizeof(c->last_error), "%s: %s", what, cudaGetErrorString(e));
    return FF_ERR_CUDA;
}

#define FF_CUDA(c, call)                                            \
    do {                                                            \
        cudaError_t e__ = (call);                                   \
        if (e__ != cudaSuccess) return ff_cuda_fail((c), e__, #call); \
    } while (0)

// launch + count + check
#define FF_LAUNCH(c, kernel, grid, block, smem, ...)                          \
    do {                                                                      \
        kernel<<<(grid), (block), (smem), (c)->stream>>>(__VA_ARGS__);        \
        (c)->launches++;                                                      \
        cudaError_t e__ = cudaGetLastError();                                 \
        if (e__ != cudaSuccess) return ff_cuda_fail((c), e__, #kernel);       \
    } while (0)

static inline void ff_phase_begin(ff_ctx* c, int ph)
{
    if (c->timing_enabled) cudaEventRecord(c->ev[ph][0], c->stream);
}
static inline void ff_phase_end(ff_ctx* c, int ph)
{
    if (c->timing_enabled) { cudaEventRecord(c->ev[ph][1], c->stream); c->ev_valid[ph] = 1; }
}

// ---- phase launchers implemented in the other .cu files -------------------------
int ff_launch_bbox_keys(ff_ctx* c, const float* pos);
int ff_launch_sort(ff_ctx* c, const float* pos);
int ff_launch_build(ff_ctx* c);
int ff_launch_moments(ff_ctx* c, const float* mom);
int ff_launch_walk(ff_ctx* c, float* H_out, float* F_out, int group_begin = 0, int group_end = -1);
int ff_launch_direct(ff_ctx* c, const float* pos, const float* mom, int64_t n, float* H_out, float* F_out,
                     float lj_eps = 0.0f, float lj_sigma = 1.0f, float lj_cutoff = 0.0f);   // lj_eps != 0: F_out = f^dip + f^sr
int ff_launch_probe(ff_ctx* c, int kind, int iters, double* tflops);
int ff_launch_lj(ff_ctx* c, int64_t n, const ff_step_params* p, cudaStream_t stream);   // -> c->step_fsr (needs the tree)
int ff_launch_integrate(ff_ctx* c, float* pos, float* vel, float* mom, float* angvel, int64_t n,
                        const ff_step_params* p, uint64_t step_index, bool with_fsr);

// ---- checked build (-DFF_CHECKED): device-side index and bound checks of every kernel --------------------------
// compute-sanitizer is not available on every machine this runs on; the checked library is what
// tests/sanitizer_smoke.py runs against instead.  A failed check sets the sticky error flag (first one wins) and the
// kernel carries on; the release build compiles the checks away.
#ifdef FF_CHECKED
#define FF_CHECK(g, cond)                                                                    \
    do {                                                                                     \
        if (!(cond) && atomicCAS(&(g)->error, 0, (int32_t)FF_ERR_CHECK) == 0) (g)->check_line = __LINE__; \
    } while (0)
#else
#define FF_CHECK(g, cond) do { } while (0)
#endif

// ---- small device helpers --------------------------------------------------------
__device__ __forceinline__ uint32_t ff_f2ord(float f)
{
    uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float ff_ord2f(uint32_t o)
{
    return __uint_as_float((o & 0x80000000u) ? (o & 0x7fffffffu) : ~o);
}
__device__ __forceinline__ int ff_lane() { return threadIdx.x & 31; }

// the device-side state a tree build starts from (thread t of nt): empty bounding box, sort tickets and digit
// histograms at zero.  Run by ff_k_reset, and by ff_k_build for the NEXT build once the current one has consumed them.
__device__ __forceinline__ void ff_reset_globals(ff_globals* g, int t, int nt)
{
    if (t < 3) { g->bbox_ord[t] = 0xffffffffu; g->bbox_ord[4 + t] = 0u; }
    if (t < 4) g->counters[t] = 0ull;
    if (t < FF_SORT_PASSES) g->sort_ticket[t] = 0;
    if (t < FF_MAX_LEVEL) { g->level_count[t] = 0; g->level_cursor[t] = 0; }
    for (int i = t; i < FF_SORT_PASSES * FF_RADIX; i += nt) (&g->digit_hist[0][0])[i] = 0u;
}

// number of leading octant digits two 30-bit keys share (10 if equal)
__device__ __forceinline__ int ff_common_levels(uint32_t a, uint32_t b)
{
    uint32_t x = a ^ b;
    return x ? (__clz(x) - 2) / 3 : FF_MAX_LEVEL;
}
