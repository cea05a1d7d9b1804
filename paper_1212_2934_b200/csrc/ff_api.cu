// ff_api.cu -- the C ABI of include/ff.h: context, workspace carve-up, phase orchestration.
#include <math.h>
#include <new>

#include "ff_internal.cuh"

static size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// One pass over the workspace layout; with base == nullptr it only measures.
static size_t carve(ff_ctx* c, char* base, int64_t N)
{
    size_t off = 0;
    auto take = [&](size_t bytes) -> char* {
        char* p = base ? base + off : nullptr;
        off += align_up(bytes);
        return p;
    };
    size_t n = (size_t)N;
    size_t cap = 5 * n + 8;                                  // <= N/2 internal cells on each of 10 levels
    size_t sort_tiles = (n + FF_SORT_TILE - 1) / FF_SORT_TILE;
    size_t scan_tiles = (n + FF_SCAN_TILE - 1) / FF_SCAN_TILE;
    char* p;
    p = take(sizeof(ff_globals));                 if (c) c->g = (ff_globals*)p;
    for (int b = 0; b < 2; ++b) {
        p = take(n * 4);                          if (c) c->key[b] = (uint32_t*)p;
        p = take(n * 4);                          if (c) c->idx[b] = (uint32_t*)p;
    }
    p = take(n * 16);                             if (c) c->pos_s = (float4*)p;
    p = take(n * 16);                             if (c) c->mom_s = (float4*)p;
    p = take(n * 4);                              if (c) c->leaf_count = (int32_t*)p;
    p = take(n * 4);                              if (c) c->cell_base = (int32_t*)p;
    p = take((scan_tiles + 1 + FF_BUILD_MAX_BLOCKS) * 4); if (c) c->scan_blk = (uint32_t*)p;   // one word per block of ff_k_build
    p = take(sort_tiles * FF_RADIX * 4 * FF_SORT_PASSES); if (c) c->sort_status = (uint32_t*)p;
    p = take(cap * 4);                            if (c) c->cell_first = (int32_t*)p;
    p = take(cap * 4);                            if (c) c->cell_end = (int32_t*)p;
    p = take(cap * 4);                            if (c) c->cell_level = (int32_t*)p;
    p = take(cap * 4);                            if (c) c->cell_list = (int32_t*)p;
    p = take(cap * 16);                           if (c) c->cell_info = (int4*)p;
    p = take(cap * 32);                           if (c) c->cell_child = (int32_t*)p;
    p = take(cap * 16);                           if (c) c->cell_centre = (float4*)p;
    p = take(cap * 16);                           if (c) c->cell_moment = (float4*)p;
    p = take(cap * 64);                           if (c) c->cell_sums = (double*)p;
    p = take(cap * 64);                           if (c) c->cell_sums2 = (double*)p;
    p = take(cap * 32);                           if (c) c->cell_quad = (float4*)p;
    p = take((size_t)FF_DIRECT_SPLIT_ELEMS * 48); if (c) c->direct_part = (double*)p;
    for (int b = 0; b < 2; ++b) {
        p = take(n * 12);                         if (c) c->stage_pos2[b] = (float*)p;
        p = take(n * 12);                         if (c) c->stage_mom2[b] = (float*)p;
        p = take(n * 12);                         if (c) c->stage_H2[b] = (float*)p;
        p = take(n * 12);                         if (c) c->stage_F2[b] = (float*)p;
    }
    if (c) { c->stage_H = c->stage_H2[0]; c->stage_F = c->stage_F2[0]; }
    p = take(n * 12);                             if (c) c->step_fsr = (float*)p;
    if (c) c->cell_cap = (int64_t)cap;
    return off;
}

extern "C" size_t ff_workspace_bytes(int64_t N)
{
    if (N <= 0 || N > FF_MAX_N) return 0;
    return carve(nullptr, nullptr, N);
}

// everything ff_create made, in any state of completion
static void ff_teardown(ff_ctx* c)
{
    for (int ph = 0; ph < FF_N_PHASES; ++ph)
        for (int k = 0; k < 2; ++k) if (c->ev[ph][k]) cudaEventDestroy(c->ev[ph][k]);
    for (int b = 0; b < 2; ++b) {
        if (c->ev_pos[b]) cudaEventDestroy(c->ev_pos[b]);
        if (c->ev_in[b]) cudaEventDestroy(c->ev_in[b]);
        if (c->ev_done[b]) cudaEventDestroy(c->ev_done[b]);
        if (c->ev_out[b]) cudaEventDestroy(c->ev_out[b]);
    }
    if (c->ev_tree) cudaEventDestroy(c->ev_tree);
    if (c->ev_lj) cudaEventDestroy(c->ev_lj);
    if (c->in_stream) cudaStreamDestroy(c->in_stream);
    if (c->out_stream) cudaStreamDestroy(c->out_stream);
    if (c->lj_stream) cudaStreamDestroy(c->lj_stream);
    delete c;
}

extern "C" int ff_create(ff_ctx** out, int64_t N, float theta, void* workspace, size_t workspace_bytes)
{
    if (!out) return FF_ERR_INVALID_ARG;
    *out = nullptr;
    if (N <= 0 || N > FF_MAX_N || !(theta >= 0.0f) || isinf(theta)) return FF_ERR_INVALID_ARG;
    size_t need = ff_workspace_bytes(N);
    if (!workspace || workspace_bytes < need || ((uintptr_t)workspace & 255)) return FF_ERR_WORKSPACE;
    ff_ctx* c = new (std::nothrow) ff_ctx;
    if (!c) return FF_ERR_INVALID_ARG;
    memset(c, 0, sizeof(*c));
    c->N = N; c->theta = theta; c->nleaf = 1; c->group = 32;
    c->ws = (char*)workspace; c->ws_bytes = workspace_bytes;
    carve(c, c->ws, N);
    cudaError_t e = cudaGetDevice(&c->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device);
    for (int ph = 0; e == cudaSuccess && ph < FF_N_PHASES; ++ph)
        for (int k = 0; e == cudaSuccess && k < 2; ++k) e = cudaEventCreate(&c->ev[ph][k]);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->in_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->out_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) {
        // a second stream at the lowest priority the device offers.  On current NVIDIA parts that value is the one
        // every default-priority stream has as well (the caller's stream included), so nothing here puts the walk's
        // blocks first: how much of the Lennard-Jones pass lands in the walk's drain is a matter of submission timing
        int least = 0, greatest = 0;
        e = cudaDeviceGetStreamPriorityRange(&least, &greatest);
        if (e == cudaSuccess) e = cudaStreamCreateWithPriority(&c->lj_stream, cudaStreamNonBlocking, least);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_tree, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_lj, cudaEventDisableTiming);
    for (int b = 0; e == cudaSuccess && b < 2; ++b) {
        e = cudaEventCreateWithFlags(&c->ev_pos[b], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_in[b], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_done[b], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_out[b], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaMemset(c->g, 0, sizeof(ff_globals));
    if (e != cudaSuccess) { ff_teardown(c); return FF_ERR_CUDA; }
    *out = c;
    return FF_OK;
}

extern "C" int ff_destroy(ff_ctx* c)
{
    if (!c) return FF_ERR_INVALID_ARG;
    ff_device_guard guard(c);
    cudaStreamSynchronize(c->stream);
    if (c->in_stream) cudaStreamSynchronize(c->in_stream);
    if (c->out_stream) cudaStreamSynchronize(c->out_stream);
    if (c->lj_stream) cudaStreamSynchronize(c->lj_stream);
    ff_teardown(c);
    return FF_OK;
}

extern "C" int ff_set_stream(ff_ctx* c, void* cuda_stream)
{
    if (!c) return FF_ERR_INVALID_ARG;
    c->stream = (cudaStream_t)cuda_stream;
    return FF_OK;
}

extern "C" int ff_set_option(ff_ctx* c, int key, double value)
{
    if (!c) return FF_ERR_INVALID_ARG;
    switch (key) {
    case FF_OPT_THETA:
        if (!(value >= 0.0) || isinf(value)) return FF_ERR_INVALID_ARG;
        c->theta = (float)value;
        return FF_OK;
    case FF_OPT_NLEAF:
        if (!(value >= 1.0) || value > 1e9) return FF_ERR_INVALID_ARG;
        c->nleaf = (int)value;
        c->tree_built = 0;
        return FF_OK;
    case FF_OPT_COUNTERS: c->count_enabled = value != 0.0; return FF_OK;
    case FF_OPT_TIMING: c->timing_enabled = value != 0.0; return FF_OK;
    case FF_OPT_GROUP:
        if (value != 32.0 && value != 64.0) return FF_ERR_INVALID_ARG;
        if (value == 64.0 && c->order == 1) return FF_ERR_INVALID_ARG;      // the first-order walk exists for W = 32 only
        c->group = (int)value;
        return FF_OK;
    case FF_OPT_CELL_ORDER:
        if (value != 0.0 && value != 1.0) return FF_ERR_INVALID_ARG;
        if (value == 1.0 && c->group != 32) return FF_ERR_INVALID_ARG;
        c->order = (int)value;
        return FF_OK;
    default: return FF_ERR_INVALID_ARG;
    }
}

extern "C" int ff_build_tree(ff_ctx* c, const float* pos, int64_t n)
{
    ff_device_guard guard(c);
    if (!c || !pos || n <= 0 || n > c->N) return FF_ERR_INVALID_ARG;
    c->n = n;
    c->tree_built = 0;
    c->moments_valid = 0;
    int rc;
    ff_phase_begin(c, FF_PH_BBOX_KEYS);
    if ((rc = ff_launch_bbox_keys(c, pos)) != FF_OK) return rc;
    ff_phase_end(c, FF_PH_BBOX_KEYS);
    ff_phase_begin(c, FF_PH_SORT);
    if ((rc = ff_launch_sort(c, pos)) != FF_OK) return rc;
    ff_phase_end(c, FF_PH_SORT);
    ff_phase_begin(c, FF_PH_BUILD);
    if ((rc = ff_launch_build(c)) != FF_OK) return rc;
    ff_phase_end(c, FF_PH_BUILD);
    c->globals_clean = 1;                                  // ff_k_build leaves the reset state for the next build
    c->tree_built = 1;
    c->tree_pos = pos;
    return FF_OK;
}

extern "C" int ff_eval_bh(ff_ctx* c, const float* pos, const float* mom, float* H_out, float* F_out)
{
    return ff_eval_bh_range(c, pos, mom, H_out, F_out, 0, -1);
}

extern "C" int ff_eval_bh_range(ff_ctx* c, const float* pos, const float* mom, float* H_out, float* F_out,
                                int64_t group_begin, int64_t group_end)
{
    ff_device_guard guard(c);
    if (!c || !pos || !mom) return FF_ERR_INVALID_ARG;
    if (!c->tree_built) return FF_ERR_NO_TREE;
    if (pos != c->tree_pos) return FF_ERR_INVALID_ARG;     // not the array the tree was built from
    const int64_t groups = (c->n + c->group - 1) / c->group;
    if (group_end < 0) group_end = groups;
    if (group_begin < 0 || group_begin > group_end || group_end > groups) return FF_ERR_INVALID_ARG;
    int rc;
    ff_phase_begin(c, FF_PH_MOMENTS);
    if ((rc = ff_launch_moments(c, mom)) != FF_OK) return rc;
    ff_phase_end(c, FF_PH_MOMENTS);
    c->moments_valid = 1;
    c->moments_order = c->order;
    ff_phase_begin(c, FF_PH_WALK);
    if ((rc = ff_launch_walk(c, H_out, F_out, (int)group_begin, (int)group_end)) != FF_OK) return rc;
    ff_phase_end(c, FF_PH_WALK);
    return FF_OK;
}

extern "C" int ff_eval_direct(ff_ctx* c, const float* pos, const float* mom, int64_t n, float* H_out, float* F_out)
{
    ff_device_guard guard(c);
    if (!c || !pos || !mom || n <= 0 || n > c->N) return FF_ERR_INVALID_ARG;
    ff_phase_begin(c, FF_PH_DIRECT);
    int rc = ff_launch_direct(c, pos, mom, n, H_out, F_out);
    if (rc != FF_OK) return rc;
    ff_phase_end(c, FF_PH_DIRECT);
    return FF_OK;
}

// ---- *_host calls: uploads, compute and downloads on three streams, double-buffered by call parity ----
// Call i uses staging buffer b = i & 1.  Ordering (events, no host waits):
//   in_stream   wait ev_done[b] (call i-2 has finished reading buffer b) ; H2D pos -> ev_pos[b] ; H2D mom -> ev_in[b]
//   stream      wait ev_pos[b] ; tree build ; wait ev_in[b] ; wait ev_out[b] (call i-2's download has left the
//               result buffer) ; moments + walk (or the all-pairs kernel) -> ev_done[b]
//   out_stream  wait ev_done[b] ; D2H H, F -> ev_out[b]
// so that in a sequence of calls the copies of one call run under the compute of its neighbours (PCIe is full
// duplex), and inside one call the moment upload runs under the tree build.
static int host_enqueue(ff_ctx* c, const float* pos_h, const float* mom_h, int64_t n, float* H_h, float* F_h, bool bh)
{
    ff_device_guard guard(c);
    if (!c || !pos_h || !mom_h || n <= 0 || n > c->N) return FF_ERR_INVALID_ARG;
    const int b = (int)(c->host_seq & 1);
    const size_t bytes = (size_t)n * 12;
    FF_CUDA(c, cudaStreamWaitEvent(c->in_stream, c->ev_done[b], 0));
    FF_CUDA(c, cudaMemcpyAsync(c->stage_pos2[b], pos_h, bytes, cudaMemcpyHostToDevice, c->in_stream));
    FF_CUDA(c, cudaEventRecord(c->ev_pos[b], c->in_stream));
    FF_CUDA(c, cudaMemcpyAsync(c->stage_mom2[b], mom_h, bytes, cudaMemcpyHostToDevice, c->in_stream));
    FF_CUDA(c, cudaEventRecord(c->ev_in[b], c->in_stream));
    float* Hd = H_h ? c->stage_H2[b] : nullptr;
    float* Fd = F_h ? c->stage_F2[b] : nullptr;
    int rc;
    FF_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_pos[b], 0));
    if (bh) {
        if ((rc = ff_build_tree(c, c->stage_pos2[b], n)) != FF_OK) return rc;
        FF_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_in[b], 0));
        FF_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_out[b], 0));
        if ((rc = ff_eval_bh(c, c->stage_pos2[b], c->stage_mom2[b], Hd, Fd)) != FF_OK) return rc;
    } else {
        FF_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_in[b], 0));
        FF_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_out[b], 0));
        if ((rc = ff_eval_direct(c, c->stage_pos2[b], c->stage_mom2[b], n, Hd, Fd)) != FF_OK) return rc;
    }
    FF_CUDA(c, cudaEventRecord(c->ev_done[b], c->stream));
    FF_CUDA(c, cudaStreamWaitEvent(c->out_stream, c->ev_done[b], 0));
    if (H_h) FF_CUDA(c, cudaMemcpyAsync(H_h, Hd, bytes, cudaMemcpyDeviceToHost, c->out_stream));
    if (F_h) FF_CUDA(c, cudaMemcpyAsync(F_h, Fd, bytes, cudaMemcpyDeviceToHost, c->out_stream));
    FF_CUDA(c, cudaEventRecord(c->ev_out[b], c->out_stream));
    c->host_seq++;
    return FF_OK;
}

extern "C" int ff_host_sync(ff_ctx* c)
{
    ff_device_guard guard(c);
    if (!c) return FF_ERR_INVALID_ARG;
    FF_CUDA(c, cudaStreamSynchronize(c->in_stream));
    FF_CUDA(c, cudaStreamSynchronize(c->stream));
    FF_CUDA(c, cudaStreamSynchronize(c->out_stream));
    return FF_OK;
}

extern "C" int ff_eval_bh_host_async(ff_ctx* c, const float* pos_h, const float* mom_h, int64_t n, float* H_h, float* F_h)
{
    return host_enqueue(c, pos_h, mom_h, n, H_h, F_h, true);
}

extern "C" int ff_eval_bh_host(ff_ctx* c, const float* pos_h, const float* mom_h, int64_t n, float* H_h, float* F_h)
{
    int rc = host_enqueue(c, pos_h, mom_h, n, H_h, F_h, true);
    return rc != FF_OK ? rc : ff_host_sync(c);
}

extern "C" int ff_eval_direct_host(ff_ctx* c, const float* pos_h, const float* mom_h, int64_t n, float* H_h, float* F_h)
{
    int rc = host_enqueue(c, pos_h, mom_h, n, H_h, F_h, false);
    return rc != FF_OK ? rc : ff_host_sync(c);
}

extern "C" int ff_step(ff_ctx* c, float* pos, float* vel, float* mom, float* angvel, int64_t n,
                       const ff_step_params* p, uint64_t step_index)
{
    ff_device_guard guard(c);
    if (!c || !pos || !vel || !mom || !angvel || !p || n <= 0 || n > c->N) return FF_ERR_INVALID_ARG;
    if (!(p->dtau > 0.0f)) return FF_ERR_INVALID_ARG;
    // every parameter check comes before the first launch: a refused call enqueues nothing and leaves the context as it was
    const bool lj = p->lj_epsilon != 0.0f;
    if (lj && (!(p->lj_cutoff > 0.0f) || !(p->lj_sigma > 0.0f))) return FF_ERR_INVALID_ARG;
    if (p->wall_epsilon != 0.0f && (!(p->lj_cutoff > 0.0f) || !(p->wall_sigma > 0.0f))) return FF_ERR_INVALID_ARG;
    int rc;
    FF_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_out[0], 0));   // a pending download of an earlier *_host_async call
    if (p->all_pairs) {
        // the paper's All-Pairs step (Algorithm 1): h^dip, f^dip and f^sr in one pair loop, no tree
        c->n = n;
        ff_phase_begin(c, FF_PH_DIRECT);
        if ((rc = ff_launch_direct(c, pos, mom, n, c->stage_H, c->stage_F, p->lj_epsilon, p->lj_sigma, p->lj_cutoff)) != FF_OK)
            return rc;
        ff_phase_end(c, FF_PH_DIRECT);
        ff_phase_begin(c, FF_PH_STEP);                             // (f^sr is already inside stage_F)
        if ((rc = ff_launch_integrate(c, pos, vel, mom, angvel, n, p, step_index, false)) != FF_OK) return rc;
        ff_phase_end(c, FF_PH_STEP);
        c->tree_built = 0;
        return FF_OK;
    }
    // The Lennard-Jones pass needs the tree (sorted keys and positions), not the fields: it is enqueued on a second
    // stream AFTER the walk and can run beside it, in the SMs the persistent walk leaves idle while it drains
    // (about 0.17 ms at N = 2^20, profiles/r2_walk_full.md); the update waits for both.  (No priority separates the
    // two streams, see ff_create.)
    if ((rc = ff_build_tree(c, pos, n)) != FF_OK) return rc;
    if (lj) FF_CUDA(c, cudaEventRecord(c->ev_tree, c->stream));
    if ((rc = ff_eval_bh(c, pos, mom, c->stage_H, c->stage_F)) != FF_OK) return rc;
    ff_phase_begin(c, FF_PH_STEP);
    if (lj) {
        FF_CUDA(c, cudaStreamWaitEvent(c->lj_stream, c->ev_tree, 0));
        rc = ff_launch_lj(c, n, p, c->lj_stream);
        // also when the pass failed part-way: whatever it did enqueue reads the sorted keys and positions, and the
        // caller's stream must not start the next tree build (which overwrites them) before that has drained
        FF_CUDA(c, cudaEventRecord(c->ev_lj, c->lj_stream));
        FF_CUDA(c, cudaStreamWaitEvent(c->stream, c->ev_lj, 0));
        if (rc != FF_OK) return rc;
    }
    if ((rc = ff_launch_integrate(c, pos, vel, mom, angvel, n, p, step_index, lj)) != FF_OK) return rc;
    ff_phase_end(c, FF_PH_STEP);
    c->tree_built = 0;                // positions moved: the tree no longer matches
    return FF_OK;
}

// the sticky device-side error flag (FF_ERR_CAPACITY), read at a point where the stream is synchronised
static int ff_device_error(ff_ctx* c)
{
    int32_t err[2] = { 0, 0 };                             // error, check_line
    FF_CUDA(c, cudaMemcpy(err, &c->g->error, sizeof(err), cudaMemcpyDeviceToHost));
    if (err[0] == FF_ERR_CHECK) snprintf(c->last_error, sizeof(c->last_error), "device-side check failed at source line %d", err[1]);
    return err[0];
}

extern "C" int ff_get_tree(ff_ctx* c, ff_tree_view* out)
{
    ff_device_guard guard(c);
    if (!c || !out) return FF_ERR_INVALID_ARG;
    if (!c->tree_built) return FF_ERR_NO_TREE;
    FF_CUDA(c, cudaStreamSynchronize(c->stream));
    ff_globals g;
    FF_CUDA(c, cudaMemcpy(&g, c->g, sizeof(g), cudaMemcpyDeviceToHost));
    if (g.error) return ff_device_error(c);
    memset(out, 0, sizeof(*out));
    out->n = c->n; out->n_cells = g.n_cells; out->nleaf = c->nleaf;
    out->lo[0] = g.lo[0]; out->lo[1] = g.lo[1]; out->lo[2] = g.lo[2]; out->S = g.S;
    out->key = c->key[0]; out->perm = c->idx[0];
    out->pos_sorted = (const float*)c->pos_s; out->mom_sorted = (const float*)c->mom_s;
    out->cell_first = c->cell_first; out->cell_end = c->cell_end; out->cell_level = c->cell_level;
    out->child = c->cell_child; out->leaf_count = c->leaf_count;
    out->cell_centre = (const float*)c->cell_centre; out->cell_moment = (const float*)c->cell_moment;
    // only if the moments of THIS tree were computed at order 1: after an order-0 evaluation, or before any, the array
    // holds an earlier tree's tensors or nothing
    out->cell_quad = (c->moments_valid && c->moments_order == 1) ? (const float*)c->cell_quad : nullptr;
    return FF_OK;
}

extern "C" int ff_get_timings(ff_ctx* c, float ms[FF_N_PHASES])
{
    ff_device_guard guard(c);
    if (!c || !ms) return FF_ERR_INVALID_ARG;
    FF_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int ph = 0; ph < FF_N_PHASES; ++ph) {
        ms[ph] = 0.0f;
        if (c->ev_valid[ph]) {
            FF_CUDA(c, cudaEventElapsedTime(&ms[ph], c->ev[ph][0], c->ev[ph][1]));
            c->ev_valid[ph] = 0;
        }
    }
    return ff_device_error(c);
}

extern "C" int ff_get_counters(ff_ctx* c, uint64_t* n_cell, uint64_t* n_particle, uint64_t* n_mac_tests)
{
    ff_device_guard guard(c);
    if (!c) return FF_ERR_INVALID_ARG;
    FF_CUDA(c, cudaStreamSynchronize(c->stream));
    unsigned long long v[3];
    FF_CUDA(c, cudaMemcpy(v, c->g->counters, sizeof(v), cudaMemcpyDeviceToHost));
    if (n_cell) *n_cell = v[0];
    if (n_particle) *n_particle = v[1];
    if (n_mac_tests) *n_mac_tests = v[2];
    return ff_device_error(c);
}

extern "C" int ff_get_prefilter_count(ff_ctx* c, uint64_t* n_parked)
{
    ff_device_guard guard(c);
    if (!c || !n_parked) return FF_ERR_INVALID_ARG;
    FF_CUDA(c, cudaStreamSynchronize(c->stream));
    unsigned long long v;
    FF_CUDA(c, cudaMemcpy(&v, c->g->counters + 3, sizeof(v), cudaMemcpyDeviceToHost));
    *n_parked = v;
    return FF_OK;
}

extern "C" int ff_get_launch_count(ff_ctx* c, uint64_t* launches)
{
    if (!c || !launches) return FF_ERR_INVALID_ARG;
    *launches = c->launches;
    return FF_OK;
}

extern "C" int ff_measure_fp32_peak(ff_ctx* c, int iters, double* tflops)
{
    ff_device_guard guard(c);
    if (!c || !tflops) return FF_ERR_INVALID_ARG;
    return ff_launch_probe(c, FF_PROBE_FFMA, iters, tflops);
}

extern "C" int ff_measure_probe(ff_ctx* c, int kind, int iters, double* tflops)
{
    ff_device_guard guard(c);
    if (!c || !tflops) return FF_ERR_INVALID_ARG;
    return ff_launch_probe(c, kind, iters, tflops);
}

extern "C" const char* ff_error_string(int code)
{
    switch (code) {
    case FF_OK: return "ok";
    case FF_ERR_INVALID_ARG: return "invalid argument";
    case FF_ERR_WORKSPACE: return "workspace missing, too small or misaligned";
    case FF_ERR_NO_TREE: return "no tree: call ff_build_tree first";
    case FF_ERR_CAPACITY: return "cell pool capacity exceeded";
    case FF_ERR_CUDA: return "CUDA error (see ff_last_error)";
    case FF_ERR_CHECK: return "device-side check failed (checked build; see ff_last_error)";
    case FF_ERR_TOO_LARGE: return "n is beyond FF_STATIC_MAX_N, the fixed limit of ff_eval_direct_static (see ff_static_last_error)";
    default: return "unknown error code";
    }
}

extern "C" const char* ff_last_error(ff_ctx* c) { return c ? c->last_error : ""; }
