// ff_walk.cu -- a6 tree walk + a7 scatter to caller order.
//
// Paper: kernel 5 walks the octree per particle; warps hold
// spatially close particles and "the first thread of a warp" fetches cell data to
// shared memory.  That design (one cell per step, broadcast to 32 lanes) leaves
// the FP32 pipe idle during every dependent cell fetch.  Here a warp owns one
// GROUP of 32 consecutive sorted targets and splits the work in two:
//
//   list building  -- each LANE pops a DIFFERENT stack entry, tests it against the
//                     whole group (opening rule O5 of DESIGN.md) and either appends
//                     it to a shared-memory interaction ring or pushes its children;
//                     traversal cost is amortised over 32 entries per round.
//   evaluation     -- whenever 32 interactions are pending every lane evaluates them
//                     for its OWN target: a dense, branch-free loop of Eq. 11 / Eq. 12
//                      fed by broadcast float4 shared-memory reads.
//
// Both produce exactly the interaction set of the oracle's recursive walk; only
// the summation order differs.  fp32 arithmetic; the opening test uses explicit
// round-to-nearest intrinsics so it is bit-identical to the oracle's.
#include "ff_internal.cuh"

struct ff_walk_smem {
    int32_t stack[FF_WALK_STACK];
    float4 pend_pos[FF_WALK_PEND];
    float4 pend_mom[FF_WALK_PEND];
    float4 mem_pos[32];
};

// One source term of Eq. 11 (h) and Eq. 12 (f) for target (p, u).  The u_k term of
// Eq. 12 is accumulated as a scalar (sk) and multiplied by u_k once at the end.
// rinv must already be 1/|rho| (0 for a term that is to be skipped).
__device__ __forceinline__ void ff_pair_accum(float dx, float dy, float dz, float rinv, float ux, float uy, float uz,
                                              float mx, float my, float mz, float& hx, float& hy, float& hz, float& fx,
                                              float& fy, float& fz, float& sk)
{
    float rinv2 = rinv * rinv;
    float rinv3 = rinv2 * rinv;
    float r5x3 = 3.0f * (rinv3 * rinv2);                 // 3 / r^5
    float a = fmaf(mz, dz, fmaf(my, dy, mx * dx));       // u_j . rho
    float b = fmaf(uz, dz, fmaf(uy, dy, ux * dx));       // u_k . rho
    float cc = fmaf(mz, uz, fmaf(my, uy, mx * ux));      // u_j . u_k
    float ca = a * r5x3;                                 // 3 (u_j.rho) / r^5
    float cb = b * r5x3;                                 // 3 (u_k.rho) / r^5
    // h += 3 rho (u_j.rho)/r^5 - u_j / r^3
    hx = fmaf(ca, dx, hx); hy = fmaf(ca, dy, hy); hz = fmaf(ca, dz, hz);
    hx = fmaf(-rinv3, mx, hx); hy = fmaf(-rinv3, my, hy); hz = fmaf(-rinv3, mz, hz);
    // f += rho [3 (u_j.u_k) - 15 (u_j.rho)(u_k.rho)/r^2]/r^5 + u_k ca + u_j cb
    float t = (a * b) * rinv2;
    float cr = fmaf(-5.0f, t, cc) * r5x3;
    fx = fmaf(cr, dx, fx); fy = fmaf(cr, dy, fy); fz = fmaf(cr, dz, fz);
    fx = fmaf(cb, mx, fx); fy = fmaf(cb, my, fy); fz = fmaf(cb, mz, fz);
    sk += ca;
}

template <bool COUNT>
__global__ void __launch_bounds__(FF_WALK_WARPS * 32)
ff_k_walk(int n, float theta, const ff_globals* __restrict__ g, const float4* __restrict__ pos_s,
          const float4* __restrict__ mom_s, const uint32_t* __restrict__ perm,
          const int32_t* __restrict__ cell_first,
          const int32_t* __restrict__ cell_end, const int4* __restrict__ cell_child,
          const int32_t* __restrict__ leaf_count, const float4* __restrict__ centre,
          const float4* __restrict__ moment, float* __restrict__ H_out, float* __restrict__ F_out,
          unsigned long long* __restrict__ counters)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    ff_walk_smem& sm = reinterpret_cast<ff_walk_smem*>(smem_raw)[w];
    const int grp = blockIdx.x * FF_WALK_WARPS + w;
    const int g0 = grp * 32;
    if (g0 >= n) return;                                   // whole warp
    const int g1 = min(n, g0 + 32);
    const int nm = g1 - g0;
    const unsigned lt = (1u << lane) - 1u;

    // own target (lanes past the end duplicate the last member; their results are dropped)
    const int k = g0 + min(lane, nm - 1);
    const float4 pk = __ldg(pos_s + k), uk = __ldg(mom_s + k);
    const float px = pk.x, py = pk.y, pz = pk.z, ux = uk.x, uy = uk.y, uz = uk.z;
    float hx = 0.f, hy = 0.f, hz = 0.f, fx = 0.f, fy = 0.f, fz = 0.f, sk = 0.f;
    unsigned long long c_cell = 0, c_part = 0, c_mac = 0;

    sm.mem_pos[lane] = pk;
    sm.pend_pos[lane] = pk;
    sm.pend_mom[lane] = uk;
    __syncwarp();
    // the group's own members: direct terms, self skipped by index (Alg. 1 line 5)
    for (int j = 0; j < nm; ++j) {
        float4 sp = sm.pend_pos[j], sv = sm.pend_mom[j];
        float dx = px - sp.x, dy = py - sp.y, dz = pz - sp.z;
        float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        float rinv = (j == lane) ? 0.0f : rsqrtf(r2);
        ff_pair_accum(dx, dy, dz, rinv, ux, uy, uz, sv.x, sv.y, sv.z, hx, hy, hz, fx, fy, fz, sk);
    }
    if (COUNT) c_part += (unsigned long long)nm * (unsigned long long)(nm - 1);
    __syncwarp();

    const float th2 = __fmul_rn(theta, theta);
    int pend_head = 0, pend_cnt = 0;                       // warp-uniform ring state
    int sp_top = 0;                                        // warp-uniform stack size

    // evaluate `cnt` pending entries starting at pend_head for this lane's target
    auto eval = [&](int cnt) {
        __syncwarp();
        if (cnt == 32) {
#pragma unroll 8
            for (int j = 0; j < 32; ++j) {
                float4 sp = sm.pend_pos[pend_head + j], sv = sm.pend_mom[pend_head + j];
                float dx = px - sp.x, dy = py - sp.y, dz = pz - sp.z;
                float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                ff_pair_accum(dx, dy, dz, rsqrtf(r2), ux, uy, uz, sv.x, sv.y, sv.z, hx, hy, hz, fx, fy, fz, sk);
            }
        } else {
            for (int j = 0; j < cnt; ++j) {
                float4 sp = sm.pend_pos[pend_head + j], sv = sm.pend_mom[pend_head + j];
                float dx = px - sp.x, dy = py - sp.y, dz = pz - sp.z;
                float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                ff_pair_accum(dx, dy, dz, rsqrtf(r2), ux, uy, uz, sv.x, sv.y, sv.z, hx, hy, hz, fx, fy, fz, sk);
            }
        }
        __syncwarp();
    };
    // append the lanes with `take` set (data A = position, B = moment) to the ring
    auto append = [&](bool take, const float4& A, const float4& B) {
        unsigned m = __ballot_sync(FF_FULL, take);
        if (take) {
            int slot = (pend_head + pend_cnt + __popc(m & lt)) & (FF_WALK_PEND - 1);
            sm.pend_pos[slot] = A;
            sm.pend_mom[slot] = B;
        }
        pend_cnt += __popc(m);
    };
    auto drain = [&]() {
        while (pend_cnt >= 32) {
            eval(32);
            pend_head = (pend_head + 32) & (FF_WALK_PEND - 1);
            pend_cnt -= 32;
        }
    };
    // a leaf with several particles (depth cap or N_leaf > 1): the warp streams it through the ring
    auto coop_leaf = [&](int first, int cnt) {
        for (int base = first; base < first + cnt; base += 32) {
            int j = base + lane;
            bool ok = j < first + cnt && !(j >= g0 && j < g1);
            float4 A = make_float4(0.f, 0.f, 0.f, 0.f), B = A;
            if (ok) { A = __ldg(pos_s + j); B = __ldg(mom_s + j); }
            append(ok, A, B);
            if (COUNT) c_part += (unsigned long long)__popc(__ballot_sync(FF_FULL, ok)) * nm;
            drain();
        }
    };

    const int n_cells = g->n_cells;
    if (n_cells == 0) {
        coop_leaf(0, n);                                   // the root is a leaf: plain all-pairs
    } else {
        if (lane == 0) sm.stack[0] = 0;                    // root cell
        sp_top = 1;
        __syncwarp();
    }

    while (sp_top > 0) {
        // entries popped this round; bounded so that the pushes always fit (walk stack)
        int room = FF_WALK_STACK - 80 - sp_top;
        int p = min(sp_top, max(1, min(32, room / 7)));
        int32_t e = (lane < p) ? sm.stack[sp_top - 1 - lane] : FF_CHILD_EMPTY;
        sp_top -= p;
        __syncwarp();
        const bool is_cell = e >= 0;
        const bool is_part = !is_cell && e != FF_CHILD_EMPTY && !((uint32_t)e & FF_CHILD_MULTI);
        const bool is_multi = !is_cell && e != FF_CHILD_EMPTY && ((uint32_t)e & FF_CHILD_MULTI);
        const int slot = (int)((uint32_t)e & FF_CHILD_SLOT);
        float4 A = make_float4(0.f, 0.f, 0.f, 0.f), B = A;
        int first = 0, end = 0;
        if (is_cell) {
            A = __ldg(centre + e); B = __ldg(moment + e);
            first = __ldg(cell_first + e); end = __ldg(cell_end + e);
        } else if (is_part) {
            A = __ldg(pos_s + slot); B = __ldg(mom_s + slot);
        }
        // opening test of every lane's cell against all members of the group: the group accepts iff
        // s^2 < fl(th2 * d2_k) for every k, i.e. iff s^2 < fl(th2 * min_k d2_k) (rounding is monotone)
        float d2min = 3.0e38f;
#pragma unroll 8
        for (int m = 0; m < 32; ++m) {
            float4 q = sm.mem_pos[m];
            float dx = __fsub_rn(q.x, A.x), dy = __fsub_rn(q.y, A.y), dz = __fsub_rn(q.z, A.z);
            float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            d2min = fminf(d2min, d2);
        }
        const bool holds = first < g1 && end > g0;         // the cell's range holds a member: always open (Q3)
        const bool tested = is_cell && !holds;
        const bool accept_cell = tested && (A.w < __fmul_rn(th2, d2min));
        const bool open = is_cell && !accept_cell;
        const bool take = accept_cell || (is_part && !(slot >= g0 && slot < g1));
        if (COUNT) {
            c_mac += __popc(__ballot_sync(FF_FULL, tested));
            c_cell += (unsigned long long)__popc(__ballot_sync(FF_FULL, accept_cell)) * nm;
            c_part += (unsigned long long)__popc(__ballot_sync(FF_FULL, take && is_part)) * nm;
        }
        append(take, A, B);
        int4 c0 = make_int4(-1, -1, -1, -1), c1 = c0;
        if (open) { c0 = __ldg(cell_child + 2 * (size_t)e); c1 = __ldg(cell_child + 2 * (size_t)e + 1); }
        drain();                                           // overlaps the child loads
        // push the children of the opened cells
        int nch = (c0.x != -1) + (c0.y != -1) + (c0.z != -1) + (c0.w != -1) + (c1.x != -1) + (c1.y != -1) +
                  (c1.z != -1) + (c1.w != -1);
        int incl = nch;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(FF_FULL, incl, o); if (lane >= o) incl += y; }
        int total = __shfl_sync(FF_FULL, incl, 31);
        if (nch) {
            int wpos = sp_top + incl - nch;
            if (c0.x != -1) sm.stack[wpos++] = c0.x;
            if (c0.y != -1) sm.stack[wpos++] = c0.y;
            if (c0.z != -1) sm.stack[wpos++] = c0.z;
            if (c0.w != -1) sm.stack[wpos++] = c0.w;
            if (c1.x != -1) sm.stack[wpos++] = c1.x;
            if (c1.y != -1) sm.stack[wpos++] = c1.y;
            if (c1.z != -1) sm.stack[wpos++] = c1.z;
            if (c1.w != -1) sm.stack[wpos++] = c1.w;
        }
        sp_top += total;
        // multi-particle leaves met this round
        unsigned mm = __ballot_sync(FF_FULL, is_multi);
        while (mm) {
            int src = __ffs(mm) - 1;
            mm &= mm - 1;
            int s0 = __shfl_sync(FF_FULL, slot, src);
            coop_leaf(s0, __ldg(leaf_count + s0));
        }
        __syncwarp();
    }
    if (pend_cnt > 0) eval(pend_cnt);

    if (lane < nm) {
        fx = fmaf(sk, ux, fx); fy = fmaf(sk, uy, fy); fz = fmaf(sk, uz, fz);
        size_t o = (size_t)__ldg(perm + k) * 3;            // a7: back to caller order
        if (H_out) { H_out[o] = hx; H_out[o + 1] = hy; H_out[o + 2] = hz; }
        if (F_out) { F_out[o] = fx; F_out[o + 1] = fy; F_out[o + 2] = fz; }
    }
    if (COUNT) {
        if (lane == 0) {
            atomicAdd(counters + 0, c_cell);
            atomicAdd(counters + 1, c_part);
            atomicAdd(counters + 2, c_mac);
        }
    }
}

int ff_launch_walk(ff_ctx* c, float* H_out, float* F_out)
{
    int n = (int)c->n;
    int groups = (n + 31) / 32;
    int blocks = (groups + FF_WALK_WARPS - 1) / FF_WALK_WARPS;
    size_t smem = sizeof(ff_walk_smem) * FF_WALK_WARPS;
    static bool attr_set = false;
    if (!attr_set) {
        FF_CUDA(c, cudaFuncSetAttribute(ff_k_walk<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        FF_CUDA(c, cudaFuncSetAttribute(ff_k_walk<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_set = true;
    }
    if (c->count_enabled) {
        FF_CUDA(c, cudaMemsetAsync(c->g->counters, 0, sizeof(c->g->counters), c->stream));
        FF_LAUNCH(c, ff_k_walk<true>, blocks, FF_WALK_WARPS * 32, smem, n, c->theta, c->g, c->pos_s, c->mom_s,
                  c->idx[0], c->cell_first, c->cell_end, (const int4*)c->cell_child,
                  c->leaf_count, c->cell_centre, c->cell_moment, H_out, F_out, c->g->counters);
    } else {
        FF_LAUNCH(c, ff_k_walk<false>, blocks, FF_WALK_WARPS * 32, smem, n, c->theta, c->g, c->pos_s, c->mom_s,
                  c->idx[0], c->cell_first, c->cell_end, (const int4*)c->cell_child,
                  c->leaf_count, c->cell_centre, c->cell_moment, H_out, F_out, c->g->counters);
    }
    return FF_OK;
}
