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
// Blackwell specific: the evaluation and the opening test are written with the
// packed FP32 instructions of sm_100 (FFMA2 / FMUL2 / FADD2 through __ffma2_rn,
// __fmul2_rn, __fadd2_rn): one lane handles TWO sources (or two group members)
// per instruction.  The FP32 pipe does the same work, but it needs half the
// issue slots, and issue was the limiter of the scalar version (profiles/).  The
// ring therefore stores sources as PAIRS: (x0,x1,y0,y1) (z0,z1,mx0,mx1)
// (my0,my1,mz0,mz1), three broadcast LDS.128 per two sources.
//
// Both phases produce exactly the interaction set of the oracle's recursive walk;
// only the summation order differs.  fp32 arithmetic; the opening test uses
// round-to-nearest intrinsics in the oracle's operation order, so every decision
// is bit-identical to the oracle's.
#include "ff_internal.cuh"
#include "ff_pair.cuh"

#define FF_PEND_PAIRS (FF_WALK_PEND / 2)

struct ff_walk_smem {
    int32_t stack[FF_WALK_STACK];
    float4 pend[FF_PEND_PAIRS * 3];    // pair p: [3p] = x0,x1,y0,y1  [3p+1] = z0,z1,mx0,mx1  [3p+2] = my0,my1,mz0,mz1
    float4 mem_xy[16];                 // group members, pair m: x0,x1,y0,y1
    float2 mem_z[16];                  //                        z0,z1
    float4 probe_xy[FF_WALK_PROBE_PAIRS];   // probe members of the opening pre-filter, same pair layout
    float2 probe_z[FF_WALK_PROBE_PAIRS];
    float4 bb_lo, bb_hi;               // bounding box of the group's members (exact min / max)
    int32_t amb[64];                   // cells the pre-filter could not decide, waiting for the full test
};

// write one interaction (A = position, B = moment) to ring slot `slot`
__device__ __forceinline__ void ff_ring_store(ff_walk_smem& sm, int slot, const float4& A, const float4& B)
{
    float* f = reinterpret_cast<float*>(sm.pend) + (slot >> 1) * 12 + (slot & 1);
    f[0] = A.x; f[2] = A.y; f[4] = A.z; f[6] = B.x; f[8] = B.y; f[10] = B.z;
}

// one group of 32 consecutive sorted targets, walked by one warp
template <bool COUNT>
__device__ __forceinline__ void
ff_walk_group(ff_walk_smem& sm, const int grp, const int lane,
          int n, float theta, const int n_cells, const float4* __restrict__ pos_s,
          const float4* __restrict__ mom_s, const uint32_t* __restrict__ perm,
          const int32_t* __restrict__ cell_first,
          const int32_t* __restrict__ cell_end, const int4* __restrict__ cell_child,
          const int32_t* __restrict__ leaf_count, const float4* __restrict__ centre,
          const float4* __restrict__ moment, float* __restrict__ H_out, float* __restrict__ F_out,
          unsigned long long* __restrict__ counters)
{
    const int g0 = grp * 32;
    const int g1 = min(n, g0 + 32);
    const int nm = g1 - g0;
    const unsigned lt = (1u << lane) - 1u;

    // own target (lanes past the end duplicate the last member; their results are dropped)
    const int k = g0 + min(lane, nm - 1);
    const float4 pk = __ldg(pos_s + k), uk = __ldg(mom_s + k);
    ff_target2 tg;
    tg.px = ff_dup(pk.x); tg.py = ff_dup(pk.y); tg.pz = ff_dup(pk.z);
    tg.ux = ff_dup(uk.x); tg.uy = ff_dup(uk.y); tg.uz = ff_dup(uk.z);
    ff_acc2 s;
    s.hx = s.hy = s.hz = s.fx = s.fy = s.fz = s.sk = ff_dup(0.0f);
    unsigned long long c_cell = 0, c_part = 0, c_mac = 0, c_amb = 0;

    {   // group members in pair layout for the opening test; the ring's first batch = the members themselves
        float* mxy = reinterpret_cast<float*>(sm.mem_xy) + (lane >> 1) * 4 + (lane & 1);
        mxy[0] = pk.x; mxy[2] = pk.y;
        reinterpret_cast<float*>(sm.mem_z)[lane] = pk.z;
        ff_ring_store(sm, lane, pk, uk);
        // pre-filter data: exact bounding box of the members and the probe members (the members that
        // attain the box extremes -- chosen on a key that trades the 5 low bits for the lane --, the
        // first and the last).  Lanes past a ragged end hold copies of the last member, which is harmless.
        const uint32_t ox = ff_f2ord(pk.x), oy = ff_f2ord(pk.y), oz = ff_f2ord(pk.z);
        const float lox = ff_ord2f(__reduce_min_sync(FF_FULL, ox)), hix = ff_ord2f(__reduce_max_sync(FF_FULL, ox));
        const float loy = ff_ord2f(__reduce_min_sync(FF_FULL, oy)), hiy = ff_ord2f(__reduce_max_sync(FF_FULL, oy));
        const float loz = ff_ord2f(__reduce_min_sync(FF_FULL, oz)), hiz = ff_ord2f(__reduce_max_sync(FF_FULL, oz));
        if (lane == 0) {
            sm.bb_lo = make_float4(lox, loy, loz, 0.f);
            sm.bb_hi = make_float4(hix, hiy, hiz, 0.f);
        }
        const uint32_t kx = (ox & ~31u) | lane, ky = (oy & ~31u) | lane, kz = (oz & ~31u) | lane;
        int src[8];
        src[0] = __reduce_min_sync(FF_FULL, kx) & 31; src[1] = __reduce_max_sync(FF_FULL, kx) & 31;
        src[2] = __reduce_min_sync(FF_FULL, ky) & 31; src[3] = __reduce_max_sync(FF_FULL, ky) & 31;
        src[4] = __reduce_min_sync(FF_FULL, kz) & 31; src[5] = __reduce_max_sync(FF_FULL, kz) & 31;
        src[6] = 0; src[7] = 31;
#pragma unroll
        for (int t = 0; t < 2 * FF_WALK_PROBE_PAIRS; ++t)
            if (lane == src[t]) {
                float* f = reinterpret_cast<float*>(sm.probe_xy) + (t >> 1) * 4 + (t & 1);
                f[0] = pk.x; f[2] = pk.y;
                reinterpret_cast<float*>(sm.probe_z)[t] = pk.z;
            }
    }
    __syncwarp();
    // the group's own members: direct terms, self skipped by index (Alg. 1 line 5);
    // slots >= nm of a ragged last group hold copies of the last member and are masked the same way
#pragma unroll 2
    for (int jj = 0; jj < 16; ++jj) {
        const float4 q0 = sm.pend[3 * jj], q1 = sm.pend[3 * jj + 1], q2 = sm.pend[3 * jj + 2];
        float2 dx, dy, dz, r2;
        ff_pair2_geom(q0, q1, tg, dx, dy, dz, r2);
        float2 rinv;
        rinv.x = (2 * jj == lane || 2 * jj >= nm) ? 0.0f : ff_rsqrt(r2.x);
        rinv.y = (2 * jj + 1 == lane || 2 * jj + 1 >= nm) ? 0.0f : ff_rsqrt(r2.y);
        ff_pair2_accum(q1, q2, tg, dx, dy, dz, rinv, s);
    }
    if (COUNT) c_part += (unsigned long long)nm * (unsigned long long)(nm - 1);
    __syncwarp();

    const float th2 = __fmul_rn(theta, theta);
    int pend_head = 0, pend_cnt = 0;                       // warp-uniform ring state (entries)
    int sp_top = 0;                                        // warp-uniform stack size

    // evaluate `pairs` pending source pairs starting at ring entry pend_head for this lane's target
    auto eval = [&](int pairs) {
        __syncwarp();
        const float4* q = sm.pend + 3 * (pend_head >> 1);
        if (pairs == 16) {
#pragma unroll 4
            for (int jj = 0; jj < 16; ++jj) {
                const float4 q0 = q[3 * jj], q1 = q[3 * jj + 1], q2 = q[3 * jj + 2];
                float2 dx, dy, dz, r2;
                ff_pair2_geom(q0, q1, tg, dx, dy, dz, r2);
                ff_pair2_accum(q1, q2, tg, dx, dy, dz, make_float2(ff_rsqrt(r2.x), ff_rsqrt(r2.y)), s);
            }
        } else {
            for (int jj = 0; jj < pairs; ++jj) {
                const float4 q0 = q[3 * jj], q1 = q[3 * jj + 1], q2 = q[3 * jj + 2];
                float2 dx, dy, dz, r2;
                ff_pair2_geom(q0, q1, tg, dx, dy, dz, r2);
                ff_pair2_accum(q1, q2, tg, dx, dy, dz, make_float2(ff_rsqrt(r2.x), ff_rsqrt(r2.y)), s);
            }
        }
        __syncwarp();
    };
    // append the lanes with `take` set (data A = position, B = moment) to the ring
    auto append = [&](bool take, const float4& A, const float4& B) {
        unsigned m = __ballot_sync(FF_FULL, take);
        if (take) ff_ring_store(sm, (pend_head + pend_cnt + __popc(m & lt)) & (FF_WALK_PEND - 1), A, B);
        pend_cnt += __popc(m);
    };
    auto drain = [&]() {
        while (pend_cnt >= 32) {
            eval(16);
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

    if (n_cells == 0) {
        coop_leaf(0, n);                                   // the root is a leaf: plain all-pairs
    } else {
        if (lane == 0) sm.stack[0] = 0;                    // root cell
        sp_top = 1;
        __syncwarp();
    }

    int amb_cnt = 0;                                       // warp-uniform size of the ambiguous queue
    while (sp_top > 0 || amb_cnt > 0) {
        // Source of this round's entries.  Normal round: pop the stack, decide cells with the cheap
        // pre-filter, park the undecided ones in sm.amb.  Ambiguous round (32 parked, or the stack ran
        // dry): full 32-member test on parked cells.  Stack nearly full: pop one entry at a time as
        // before; parked cells wait (and, if 32 are parked already, popped cells get the full test).
        const int room = FF_WALK_STACK - 80 - sp_top;
        const bool amb_round = sp_top == 0 || (amb_cnt >= 32 && room >= FF_WALK_AMB_ROOM);
        const bool full = amb_round || amb_cnt >= 32;
        int32_t e;
        if (amb_round) {
            const int p = min(amb_cnt, 32);
            e = (lane < p) ? sm.amb[amb_cnt - 1 - lane] : FF_CHILD_EMPTY;
            amb_cnt -= p;
        } else {
            // entries popped this round; bounded so that the pushes always fit (walk stack)
            const int p = min(sp_top, max(1, min(32, room / 7)));
            e = (lane < p) ? sm.stack[sp_top - 1 - lane] : FF_CHILD_EMPTY;
            sp_top -= p;
        }
        __syncwarp();
        const bool is_cell = e >= 0;
        const bool is_part = !is_cell && e != FF_CHILD_EMPTY && !((uint32_t)e & FF_CHILD_MULTI);
        const bool is_multi = !is_cell && e != FF_CHILD_EMPTY && ((uint32_t)e & FF_CHILD_MULTI);
        const int slot = (int)((uint32_t)e & FF_CHILD_SLOT);
        float4 A = make_float4(0.f, 0.f, 0.f, 0.f), B = A;
        int first = 0, end = 0;
        if (is_cell) {
            A = __ldg(centre + e); B = __ldg(moment + e);
            if (!amb_round) { first = __ldg(cell_first + e); end = __ldg(cell_end + e); }
        } else if (is_part) {
            A = __ldg(pos_s + slot); B = __ldg(mom_s + slot);
        }
        // Opening rule O5: the group accepts a cell iff s^2 < fl(th2 * d2_k) for every member k, i.e. iff
        // s^2 < fl(th2 * min_k d2_k) (rounding is monotone), with d = fl(q - c) as fl(q + (-c)) and
        // d2 = fma(dz,dz,fma(dy,dy,fl(dx*dx))); two members per packed instruction.
        bool acc, amb = false;
        const float2 nax = ff_dup(-A.x), nay = ff_dup(-A.y), naz = ff_dup(-A.z);
        if (full) {
            float d2min = 3.0e38f;
#pragma unroll 8
            for (int m = 0; m < 16; ++m) {
                const float4 qxy = sm.mem_xy[m];
                const float2 qz = sm.mem_z[m];
                const float2 dx = __fadd2_rn(make_float2(qxy.x, qxy.y), nax);
                const float2 dy = __fadd2_rn(make_float2(qxy.z, qxy.w), nay);
                const float2 dz = __fadd2_rn(qz, naz);
                const float2 d2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
                d2min = fminf(d2min, fminf(d2.x, d2.y));
            }
            acc = A.w < __fmul_rn(th2, d2min);
        } else {
            // Pre-filter.  (1) Sure accept: every member lies in the box, so per axis |q - c| >= e_a =
            // max(lo_a - c_a, c_a - hi_a, 0) and every exact d2_k >= e.e; the fp32 values of both sides
            // are within 6 ulp of their exact ones and the products within 1, so a margin of 2^-19
            // (0.999998f) makes "s^2 < th2 * e.e * margin" imply the exact test of every member.
            // (2) Sure open: the exact test of a probe member fails.  Anything else is parked.
            const float4 lo = sm.bb_lo, hi = sm.bb_hi;
            const float ex = fmaxf(fmaxf(lo.x - A.x, A.x - hi.x), 0.f);
            const float ey = fmaxf(fmaxf(lo.y - A.y, A.y - hi.y), 0.f);
            const float ez = fmaxf(fmaxf(lo.z - A.z, A.z - hi.z), 0.f);
            const float e2 = fmaf(ez, ez, fmaf(ey, ey, ex * ex));
            acc = A.w < th2 * e2 * 0.999998f;
            float d2min = 3.0e38f;
#pragma unroll
            for (int m = 0; m < FF_WALK_PROBE_PAIRS; ++m) {
                const float4 qxy = sm.probe_xy[m];
                const float2 qz = sm.probe_z[m];
                const float2 dx = __fadd2_rn(make_float2(qxy.x, qxy.y), nax);
                const float2 dy = __fadd2_rn(make_float2(qxy.z, qxy.w), nay);
                const float2 dz = __fadd2_rn(qz, naz);
                const float2 d2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
                d2min = fminf(d2min, fminf(d2.x, d2.y));
            }
            amb = !acc && (A.w < __fmul_rn(th2, d2min));
        }
        const bool holds = first < g1 && end > g0;         // the cell's range holds a member: always open (Q3)
        const bool tested = is_cell && !holds;
        const bool accept_cell = tested && acc;
        const bool park = tested && amb;
        const bool open = is_cell && !accept_cell && !park;
        const bool take = accept_cell || (is_part && !(slot >= g0 && slot < g1));
        if (COUNT) {
            c_mac += __popc(__ballot_sync(FF_FULL, tested && !amb_round));
            c_cell += (unsigned long long)__popc(__ballot_sync(FF_FULL, accept_cell)) * nm;
            c_part += (unsigned long long)__popc(__ballot_sync(FF_FULL, take && is_part)) * nm;
            c_amb += __popc(__ballot_sync(FF_FULL, park));
        }
        if (!full) {
            const unsigned pm = __ballot_sync(FF_FULL, park);
            if (park) sm.amb[amb_cnt + __popc(pm & lt)] = e;
            amb_cnt += __popc(pm);
        }
        append(take, A, B);
        int4 c0 = make_int4(-1, -1, -1, -1), c1 = c0;
        if (open) { c0 = __ldg(cell_child + 2 * (size_t)e); c1 = __ldg(cell_child + 2 * (size_t)e + 1); }
        const int lcnt = is_multi ? __ldg(leaf_count + slot) : 0;
        drain();                                           // overlaps the child loads
        // a bucket leaf of up to eight particles (N_leaf > 1) is expanded like an opened cell: its particles go
        // back on the stack as single-particle entries and are handled 32 at a time in the coming rounds
        const bool small_leaf = is_multi && lcnt <= 8;
        if (small_leaf) {
            const int32_t p0 = (int32_t)(FF_CHILD_LEAF1 | (uint32_t)slot);
            c0 = make_int4(p0, lcnt > 1 ? p0 + 1 : -1, lcnt > 2 ? p0 + 2 : -1, lcnt > 3 ? p0 + 3 : -1);
            c1 = make_int4(lcnt > 4 ? p0 + 4 : -1, lcnt > 5 ? p0 + 5 : -1, lcnt > 6 ? p0 + 6 : -1, lcnt > 7 ? p0 + 7 : -1);
        }
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
        unsigned mm = __ballot_sync(FF_FULL, is_multi && !small_leaf);
        while (mm) {
            int src = __ffs(mm) - 1;
            mm &= mm - 1;
            coop_leaf(__shfl_sync(FF_FULL, slot, src), __shfl_sync(FF_FULL, lcnt, src));
        }
        __syncwarp();
    }
    if (pend_cnt > 0) {
        // pad an odd tail with a copy of the last entry's position carrying a zero moment: every term
        // of Eq. 11-12 is linear in u_j, so the pad contributes exactly 0 and stays finite
        if (pend_cnt & 1) {
            __syncwarp();
            if (lane == 0) {
                const float* f = reinterpret_cast<const float*>(sm.pend);
                int last = (pend_head + pend_cnt - 1) & (FF_WALK_PEND - 1);
                const float* src = f + (last >> 1) * 12 + (last & 1);
                float4 A = make_float4(src[0], src[2], src[4], 0.f);
                ff_ring_store(sm, (last + 1) & (FF_WALK_PEND - 1), A, make_float4(0.f, 0.f, 0.f, 0.f));
            }
        }
        eval((pend_cnt + 1) >> 1);
    }

    if (lane < nm) {
        // fold the even / odd halves; f = fv + sk u_k
        const float sk = s.sk.x + s.sk.y;
        const float fx = fmaf(sk, uk.x, s.fx.x + s.fx.y), fy = fmaf(sk, uk.y, s.fy.x + s.fy.y),
                    fz = fmaf(sk, uk.z, s.fz.x + s.fz.y);
        size_t o = (size_t)__ldg(perm + k) * 3;            // a7: back to caller order
        if (H_out) { H_out[o] = s.hx.x + s.hx.y; H_out[o + 1] = s.hy.x + s.hy.y; H_out[o + 2] = s.hz.x + s.hz.y; }
        if (F_out) { F_out[o] = fx; F_out[o + 1] = fy; F_out[o + 2] = fz; }
    }
    if (COUNT) {
        if (lane == 0) {
            atomicAdd(counters + 0, c_cell);
            atomicAdd(counters + 1, c_part);
            atomicAdd(counters + 2, c_mac);
            atomicAdd(counters + 3, c_amb);
        }
    }
}

// Persistent launch: every warp fetches the next group from a device-wide counter (g->walk_next,
// zeroed by the last cell-moment launch), so no SM idles while one block's slowest group finishes
// and consecutive (spatially adjacent) groups run at the same time and share cells in L1/L2.
template <bool COUNT>
__global__ void __launch_bounds__(FF_WALK_WARPS * 32, FF_WALK_MINB)
ff_k_walk(int n, int group_begin, int group_end, float theta, ff_globals* __restrict__ g, const float4* __restrict__ pos_s,
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
    const int groups = group_end;                          // groups [group_begin, group_end) of the sorted order
    const int n_cells = g->n_cells;
    for (;;) {
        int grp = 0;
        if (lane == 0) grp = group_begin + atomicAdd(&g->walk_next, 1);
        grp = __shfl_sync(FF_FULL, grp, 0);
        if (grp >= groups) break;
        ff_walk_group<COUNT>(sm, grp, lane, n, theta, n_cells, pos_s, mom_s, perm, cell_first, cell_end, cell_child,
                             leaf_count, centre, moment, H_out, F_out, counters);
        __syncwarp();
    }
}

int ff_launch_walk(ff_ctx* c, float* H_out, float* F_out, int group_begin, int group_end)
{
    int n = (int)c->n;
    if (group_end < 0) group_end = (n + 31) / 32;
    int groups = group_end - group_begin;
    if (groups <= 0) return FF_OK;
    size_t smem = sizeof(ff_walk_smem) * FF_WALK_WARPS;
    int* per_sm = c->occ_walk;                             // per context: contexts may live on different devices
    if (!per_sm[0]) {
        FF_CUDA(c, cudaFuncSetAttribute(ff_k_walk<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        FF_CUDA(c, cudaFuncSetAttribute(ff_k_walk<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        FF_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[0], ff_k_walk<false>, FF_WALK_WARPS * 32, smem));
        FF_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm[1], ff_k_walk<true>, FF_WALK_WARPS * 32, smem));
        if (per_sm[0] < 1 || per_sm[1] < 1) return FF_ERR_CUDA;
    }
    int cnt = c->count_enabled ? 1 : 0;
    int blocks = min(c->num_sms * per_sm[cnt], (groups + FF_WALK_WARPS - 1) / FF_WALK_WARPS);
    if (cnt) {
        FF_CUDA(c, cudaMemsetAsync(c->g->counters, 0, sizeof(c->g->counters), c->stream));
        FF_LAUNCH(c, ff_k_walk<true>, blocks, FF_WALK_WARPS * 32, smem, n, group_begin, group_end, c->theta, c->g, c->pos_s, c->mom_s,
                  c->idx[0], c->cell_first, c->cell_end, (const int4*)c->cell_child,
                  c->leaf_count, c->cell_centre, c->cell_moment, H_out, F_out, c->g->counters);
    } else {
        FF_LAUNCH(c, ff_k_walk<false>, blocks, FF_WALK_WARPS * 32, smem, n, group_begin, group_end, c->theta, c->g, c->pos_s, c->mom_s,
                  c->idx[0], c->cell_first, c->cell_end, (const int4*)c->cell_child,
                  c->leaf_count, c->cell_centre, c->cell_moment, H_out, F_out, c->g->counters);
    }
    return FF_OK;
}
