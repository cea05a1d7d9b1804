// ff_walk.cu -- a6 tree walk + a7 scatter to caller order.
//
// Paper: kernel 5 walks the octree per particle; warps hold
// spatially close particles and "the first thread of a warp" fetches cell data to
// shared memory.  That design (one cell per step, broadcast to 32 lanes) leaves
// the FP32 pipe idle during every dependent cell fetch.  Here a warp owns one
// GROUP of W consecutive sorted targets (W = 32 by default, 64 as an option:
// DESIGN.md reading Q2) and splits the work in two:
//
//   list building  -- each LANE pops a DIFFERENT stack entry, tests it against the
//                     whole group (opening rule O5 of DESIGN.md) and either appends
//                     it to a shared-memory interaction ring or pushes its children;
//                     traversal cost is amortised over 32 entries per round.
//   evaluation     -- whenever 32 interactions are pending every lane evaluates them
//                     for its OWN TWO targets: a dense, branch-free loop of Eq. 11 /
//                     Eq. 12 fed by broadcast shared-memory reads.
//
// Blackwell specific: the evaluation and the opening test are written with the
// packed FP32 instructions of sm_100 (FFMA2 / FMUL2 / FADD2 through __ffma2_rn,
// __fmul2_rn, __fadd2_rn).  Every lane holds TWO targets in the halves of its
// register pairs and evaluates one source against both per instruction
// (ff_pair.cuh).  W = 32: lanes l and l + 16 hold the same two targets (2l, 2l + 1)
// and split the sources of a batch between them (even / odd ring entries); the
// two partial sums are added with one shuffle per accumulator at the end.
// W = 64: lane l holds targets 2l and 2l + 1 and every lane evaluates every source.
//
// Both phases produce exactly the interaction set of the oracle's recursive walk;
// only the summation order differs.  fp32 arithmetic; the opening test uses
// round-to-nearest intrinsics in the oracle's operation order, so every decision
// is bit-identical to the oracle's.
#include "ff_internal.cuh"
#include "ff_pair.cuh"

template <int W, bool QUAD>
struct ff_walk_smem {
    int32_t stack[FF_WALK_STACK];
    float4 pendA[FF_WALK_PEND];        // ring entry e: x, y, z, mx
    float2 pendB[FF_WALK_PEND];        //               my, mz
    float4 pendQ0[QUAD ? FF_WALK_PEND : 1];   // FF_OPT_CELL_ORDER = 1: the cell tensor Dxx, Dyy, Dzz, Dxy
    float2 pendQ1[QUAD ? FF_WALK_PEND : 1];   //                                         Dxz, Dyz  (0 for a particle)
    float4 mem_xy[W / 2];              // group members in pairs (pair m = members 2m, 2m + 1): x0,x1,y0,y1
    float2 mem_z[W / 2];               //                                                        z0,z1
    float4 mem_uxy[W / 2];             // their moments, same layout: ux0,ux1,uy0,uy1
    float2 mem_uz[W / 2];              //                             uz0,uz1
    float4 probe_xy[FF_WALK_PROBE_PAIRS];   // probe members of the opening pre-filter, same pair layout
    float2 probe_z[FF_WALK_PROBE_PAIRS];
    float4 bb_lo, bb_hi;               // bounding box of the group's members (exact min / max)
    int32_t amb[64];                   // cells the pre-filter could not decide, waiting for the full test
};

// one group of W consecutive sorted targets, walked by one warp
template <int W, bool COUNT, bool BUCKET, bool QUAD>
__device__ __forceinline__ void
ff_walk_group(ff_walk_smem<W, QUAD>& sm, const int grp, const int lane,
          int n, float theta, const int n_cells, const float4* __restrict__ pos_s,
          const float4* __restrict__ mom_s, const uint32_t* __restrict__ perm,
          const int4* __restrict__ cell_info, const int4* __restrict__ cell_child,
          const int32_t* __restrict__ leaf_count, const float4* __restrict__ centre,
          const float4* __restrict__ moment, const float4* __restrict__ quad, float* __restrict__ H_out,
          float* __restrict__ F_out, unsigned long long* __restrict__ counters, ff_globals* __restrict__ g)
{
    constexpr int ST = (W == 32) ? 2 : 1;                  // ring entries per evaluation step of one lane
    constexpr int BATCH_ITERS = FF_WALK_BATCH / ST;        // evaluation steps per batch of ring entries
    const int g0 = grp * W;
    const int g1 = min(n, g0 + W);
    const int nm = g1 - g0;
    const unsigned lt = (1u << lane) - 1u;
    const int half = (W == 32) ? (lane >> 4) : 0;          // W = 32: this lane takes the even (0) or odd (1) entries
    const int ti = (W == 32) ? (lane & 15) : lane;         // the lane's two targets are the ADJACENT members 2 ti, 2 ti + 1
    const int i0 = 2 * ti, i1 = 2 * ti + 1;
    const int k0 = g0 + min(i0, nm - 1), k1 = g0 + min(i1, nm - 1);
    unsigned long long c_cell = 0, c_part = 0, c_mac = 0, c_amb = 0;

    {   // Group members -> shared memory in pair layout (pair m = members 2m, 2m + 1) for the opening test and for the
        // lanes' own target registers; the ring's first batch(es) = the members themselves.  Members past a ragged
        // end duplicate the last member (their results are dropped).
        auto put_member = [&](int i, const float4& p, const float4& u) {
            float* mxy = reinterpret_cast<float*>(sm.mem_xy) + (i >> 1) * 4 + (i & 1);
            mxy[0] = p.x; mxy[2] = p.y;
            reinterpret_cast<float*>(sm.mem_z)[i] = p.z;
            float* uxy = reinterpret_cast<float*>(sm.mem_uxy) + (i >> 1) * 4 + (i & 1);
            uxy[0] = u.x; uxy[2] = u.y;
            reinterpret_cast<float*>(sm.mem_uz)[i] = u.z;
            sm.pendA[i] = make_float4(p.x, p.y, p.z, u.x);
            sm.pendB[i] = make_float2(u.y, u.z);
        };
        (void)quad;
        const int ma = g0 + min(lane, nm - 1), mb = g0 + min(lane + 32, nm - 1);
        const float4 pa = __ldg(pos_s + ma), ua = __ldg(mom_s + ma);
        const float4 pb = (W == 64) ? __ldg(pos_s + mb) : pa, ub = (W == 64) ? __ldg(mom_s + mb) : ua;
        put_member(lane, pa, ua);
        if (W == 64) put_member(lane + 32, pb, ub);
        // pre-filter data: exact bounding box of the members and the probe members (the members that attain the x
        // and y extremes of the box, chosen on a key that trades the low bits for the member index)
        const uint32_t ox = min(ff_f2ord(pa.x), ff_f2ord(pb.x)), oy = min(ff_f2ord(pa.y), ff_f2ord(pb.y)),
                       oz = min(ff_f2ord(pa.z), ff_f2ord(pb.z));
        const uint32_t Ox = max(ff_f2ord(pa.x), ff_f2ord(pb.x)), Oy = max(ff_f2ord(pa.y), ff_f2ord(pb.y)),
                       Oz = max(ff_f2ord(pa.z), ff_f2ord(pb.z));
        const float lox = ff_ord2f(__reduce_min_sync(FF_FULL, ox)), hix = ff_ord2f(__reduce_max_sync(FF_FULL, Ox));
        const float loy = ff_ord2f(__reduce_min_sync(FF_FULL, oy)), hiy = ff_ord2f(__reduce_max_sync(FF_FULL, Oy));
        const float loz = ff_ord2f(__reduce_min_sync(FF_FULL, oz)), hiz = ff_ord2f(__reduce_max_sync(FF_FULL, Oz));
        if (lane == 0) {
            sm.bb_lo = make_float4(lox, loy, loz, 0.f);
            sm.bb_hi = make_float4(hix, hiy, hiz, 0.f);
        }
        static_assert(FF_WALK_PROBE_PAIRS == 2, "four probe members: the x and y extremes");
        constexpr uint32_t IM = W - 1;                     // member index in the low bits of the key
        auto key = [&](float a, int i) { return (ff_f2ord(a) & ~IM) | (uint32_t)i; };
        const int s0 = __reduce_min_sync(FF_FULL, min(key(pa.x, lane), key(pb.x, lane + W - 32))) & IM;
        const int s1 = __reduce_max_sync(FF_FULL, max(key(pa.x, lane), key(pb.x, lane + W - 32))) & IM;
        const int s2 = __reduce_min_sync(FF_FULL, min(key(pa.y, lane), key(pb.y, lane + W - 32))) & IM;
        const int s3 = __reduce_max_sync(FF_FULL, max(key(pa.y, lane), key(pb.y, lane + W - 32))) & IM;
        __syncwarp();
        if (lane < 2 * FF_WALK_PROBE_PAIRS) {
            const int m = lane == 0 ? s0 : lane == 1 ? s1 : lane == 2 ? s2 : s3;
            const float* mxy = reinterpret_cast<const float*>(sm.mem_xy) + (m >> 1) * 4 + (m & 1);
            float* f = reinterpret_cast<float*>(sm.probe_xy) + (lane >> 1) * 4 + (lane & 1);
            f[0] = mxy[0]; f[2] = mxy[2];
            reinterpret_cast<float*>(sm.probe_z)[lane] = reinterpret_cast<const float*>(sm.mem_z)[m];
        }
    }
    // own targets: read back from the pair layout with vector loads, so that every target value sits in an aligned
    // register pair from the start (pairs assembled from separately loaded registers are rebuilt by ptxas with two
    // MOVs per use inside the evaluation loop)
    ff_target2 tg;
    {
        const float4 xy = sm.mem_xy[ti], uxy = sm.mem_uxy[ti];
        tg.px = make_float2(xy.x, xy.y); tg.py = make_float2(xy.z, xy.w); tg.pz = sm.mem_z[ti];
        tg.ux = make_float2(uxy.x, uxy.y); tg.uy = make_float2(uxy.z, uxy.w); tg.uz = sm.mem_uz[ti];
    }
    ff_acc2 s;                                             // QUAD: vector form of the force + cell-tensor sums
    ff_acc2_zero(s);
    ff_accq2 sq;
    ff_accq2_zero(sq);
    ff_accg2 sg;                                           // otherwise: field + force-gradient tensor (ff_pair.cuh)
    ff_accg2_zero(sg);
    __syncwarp();
    // the group's own members: direct terms, self skipped by index (Alg. 1 line 5);
    // slots >= nm of a ragged last group hold copies of the last member and are masked the same way
#pragma unroll 2
    for (int jj = 0; jj < W / ST; ++jj) {
        const int j = ST * jj + half;
        const float4 A = sm.pendA[j];
        const float2 B = sm.pendB[j];
        float2 dx, dy, dz, r2;
        ff_pair2_geom(A, tg, dx, dy, dz, r2);
        float2 rinv;
        rinv.x = (j == i0 || j >= nm) ? 0.0f : ff_rsqrt(r2.x);
        rinv.y = (j == i1 || j >= nm) ? 0.0f : ff_rsqrt(r2.y);
        if (QUAD) ff_pair2_accum(A, B, tg, dx, dy, dz, rinv, s);
        else ff_pair2g_accum(A, B, dx, dy, dz, rinv, sg);
    }
    if (COUNT) c_part += (unsigned long long)nm * (unsigned long long)(nm - 1);
    __syncwarp();

    const float th2 = __fmul_rn(theta, theta);
    int pend_head = 0, pend_cnt = 0;                       // warp-uniform ring state (entries); head is 0 or FF_WALK_BATCH
    int sp_top = 0;                                        // warp-uniform stack size

    // evaluate `iters` steps of this lane starting at ring entry pend_head (W = 32: entries head + 2 i + half)
    auto eval = [&](int iters) {
        __syncwarp();
        const float4* qa = sm.pendA + pend_head + half;
        const float2* qb = sm.pendB + pend_head + half;
        if (QUAD) {
            const float4* q0 = sm.pendQ0 + pend_head + half;
            const float2* q1 = sm.pendQ1 + pend_head + half;
            if (iters == BATCH_ITERS) {
#pragma unroll 2
                for (int i = 0; i < BATCH_ITERS; ++i) ff_pair2_quad(qa[ST * i], qb[ST * i], q0[ST * i], q1[ST * i], tg, s, sq);
            } else {
                for (int i = 0; i < iters; ++i) ff_pair2_quad(qa[ST * i], qb[ST * i], q0[ST * i], q1[ST * i], tg, s, sq);
            }
        } else if (iters == BATCH_ITERS) {
#pragma unroll 4
            for (int i = 0; i < BATCH_ITERS; ++i) ff_pair2g(qa[ST * i], qb[ST * i], tg, sg);
        } else {
            for (int i = 0; i < iters; ++i) ff_pair2g(qa[ST * i], qb[ST * i], tg, sg);
        }
        __syncwarp();
    };
    // append the lanes with `take` set (A = x, y, z, mx; B = my, mz) to the ring
    // (QUAD: `first` marks the accepted cells of a round; they go in front of the round's particles, so that
    // neighbouring ring entries are of one kind and ff_pair2_quad's skip of the first-order block seldom diverges)
    auto append = [&](bool take, const float4& A, const float2& B, const float4& Q0, const float2& Q1, bool first = false) {
        const unsigned m = __ballot_sync(FF_FULL, take);
        int rank = __popc(m & lt);
        if (QUAD) {
            const unsigned mf = __ballot_sync(FF_FULL, take && first);
            rank = first ? __popc(mf & lt) : __popc(mf) + __popc(m & ~mf & lt);
        }
        if (take) {
            const int slot = (pend_head + pend_cnt + rank) & (FF_WALK_PEND - 1);
            sm.pendA[slot] = A;
            sm.pendB[slot] = B;
            if (QUAD) { sm.pendQ0[slot] = Q0; sm.pendQ1[slot] = Q1; }
        }
        pend_cnt += __popc(m);
        FF_CHECK(g, pend_cnt <= FF_WALK_PEND);
    };
    auto drain = [&]() {
        while (pend_cnt >= FF_WALK_BATCH) {
            eval(BATCH_ITERS);
            pend_head ^= FF_WALK_BATCH;
            pend_cnt -= FF_WALK_BATCH;
        }
    };
    // a leaf with several particles (depth cap, or N_leaf > 8): the warp streams it through the ring
    auto coop_leaf = [&](int first, int cnt) {
        for (int base = first; base < first + cnt; base += 32) {
            const int j = base + lane;
            const bool ok = j < first + cnt && !(j >= g0 && j < g1);
            float4 A = make_float4(0.f, 0.f, 0.f, 0.f), B = A;
            if (ok) { A = __ldg(pos_s + j); B = __ldg(mom_s + j); }
            append(ok, make_float4(A.x, A.y, A.z, B.x), make_float2(B.y, B.z), make_float4(0.f, 0.f, 0.f, 0.f),
                   make_float2(0.f, 0.f));
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
        // dry): full W-member test on parked cells.  Stack nearly full: pop one entry at a time as
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
        FF_CHECK(g, !is_cell || e < n_cells);
        FF_CHECK(g, is_cell || e == FF_CHILD_EMPTY || (int)((uint32_t)e & FF_CHILD_SLOT) < n);
        const bool is_leaf = !is_cell && e != FF_CHILD_EMPTY;
        const bool is_multi = is_leaf && ((uint32_t)e & FF_CHILD_MULTI);
        const bool is_part = is_leaf && !is_multi;
        const int slot = (int)((uint32_t)e & FF_CHILD_SLOT);
        float4 A = make_float4(0.f, 0.f, 0.f, 0.f), B = A;
        int4 info = make_int4(0, 0, 0, 0);                 // first, end, number of children
        if (is_cell) {
            A = __ldg(centre + e); B = __ldg(moment + e); info = __ldg(cell_info + e);
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
            for (int m = 0; m < W / 2; ++m) {
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
        const bool holds = info.x < g1 && info.y > g0;     // the cell's range holds a member: always open (Q3)
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
            FF_CHECK(g, amb_cnt + __popc(pm) <= 64);
            if (park) sm.amb[amb_cnt + __popc(pm & lt)] = e;
            amb_cnt += __popc(pm);
        }
        {
            float4 Q0 = make_float4(0.f, 0.f, 0.f, 0.f);
            float2 Q1 = make_float2(0.f, 0.f);
            if (QUAD && accept_cell) {
                Q0 = __ldg(quad + 2 * (size_t)e);
                const float4 t4 = __ldg(quad + 2 * (size_t)e + 1);
                Q1 = make_float2(t4.x, t4.y);
            }
            append(take, make_float4(A.x, A.y, A.z, B.x), make_float2(B.y, B.z), Q0, Q1, accept_cell);
        }
        // the children of an opened cell: the non-empty sub-cells, compacted to the front of its eight links
        int4 c0 = make_int4(-1, -1, -1, -1), c1 = c0;
        int nch = 0;
        if (open) {
            c0 = __ldg(cell_child + 2 * (size_t)e); c1 = __ldg(cell_child + 2 * (size_t)e + 1);
            nch = info.z;
        }
        const int lcnt = is_multi ? __ldg(leaf_count + slot) : 0;
        drain();                                           // overlaps the child loads
        bool stream_leaf = is_multi;
        if (BUCKET) {
            // a bucket leaf of up to eight particles (N_leaf > 1) is expanded like an opened cell: its particles go
            // back on the stack as single-particle entries and are handled 32 at a time in the coming rounds
            if (is_multi && lcnt <= 8) {
                const int32_t q0 = (int32_t)(FF_CHILD_LEAF1 | (uint32_t)slot);
                c0 = make_int4(q0, q0 + 1, q0 + 2, q0 + 3);
                c1 = make_int4(q0 + 4, q0 + 5, q0 + 6, q0 + 7);
                nch = lcnt;
                stream_leaf = false;
            }
        }
        // push the children of the opened cells
        int incl = nch;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { int y = __shfl_up_sync(FF_FULL, incl, o); if (lane >= o) incl += y; }
        const int total = __shfl_sync(FF_FULL, incl, 31);
        FF_CHECK(g, sp_top + total <= FF_WALK_STACK && nch <= 8);
        {
            int32_t* w = sm.stack + (sp_top + incl - nch);
            if (nch > 0) w[0] = c0.x;
            if (nch > 1) w[1] = c0.y;
            if (nch > 2) w[2] = c0.z;
            if (nch > 3) w[3] = c0.w;
            if (nch > 4) w[4] = c1.x;
            if (nch > 5) w[5] = c1.y;
            if (nch > 6) w[6] = c1.z;
            if (nch > 7) w[7] = c1.w;
        }
        sp_top += total;
        // multi-particle leaves met this round
        unsigned mm = __ballot_sync(FF_FULL, stream_leaf);
        while (mm) {
            const int src = __ffs(mm) - 1;
            mm &= mm - 1;
            coop_leaf(__shfl_sync(FF_FULL, slot, src), __shfl_sync(FF_FULL, lcnt, src));
        }
        __syncwarp();
    }
    if (pend_cnt > 0) {
        // W = 32: the two half-warps take the even / odd entries; an odd tail is padded with a copy of the last
        // entry's position carrying a zero moment: every term of Eq. 11-12 is linear in u_j, so the pad contributes
        // exactly 0 and stays finite
        if (W == 32 && (pend_cnt & 1)) {
            __syncwarp();
            if (lane == 0) {
                const float4 last = sm.pendA[pend_head + pend_cnt - 1];
                sm.pendA[pend_head + pend_cnt] = make_float4(last.x, last.y, last.z, 0.f);
                sm.pendB[pend_head + pend_cnt] = make_float2(0.f, 0.f);
                if (QUAD) {
                    sm.pendQ0[pend_head + pend_cnt] = make_float4(0.f, 0.f, 0.f, 0.f);
                    sm.pendQ1[pend_head + pend_cnt] = make_float2(0.f, 0.f);
                }
            }
        }
        eval((pend_cnt + ST - 1) / ST);
    }

    // W = 32: lanes l and l + 16 hold partial sums of the same two targets
    if (W == 32) {
#define FF_FOLD(v) v.x += __shfl_xor_sync(FF_FULL, v.x, 16); v.y += __shfl_xor_sync(FF_FULL, v.y, 16)
        if (QUAD) { FF_FOLD(s.hx); FF_FOLD(s.hy); FF_FOLD(s.hz); FF_FOLD(s.fx); FF_FOLD(s.fy); FF_FOLD(s.fz); FF_FOLD(s.sk); }
        else {
            FF_FOLD(sg.hx); FF_FOLD(sg.hy); FF_FOLD(sg.hz); FF_FOLD(sg.txx); FF_FOLD(sg.tyy); FF_FOLD(sg.tzz);
            FF_FOLD(sg.gxy); FF_FOLD(sg.gxz); FF_FOLD(sg.gyz);
        }
        if (QUAD) { FF_FOLD(sq.gxx); FF_FOLD(sq.gyy); FF_FOLD(sq.gzz); FF_FOLD(sq.gxy); FF_FOLD(sq.gxz); FF_FOLD(sq.gyz); }
#undef FF_FOLD
    }
    if (QUAD) {
        // df also holds -2 (sum_j c1 D_j) u_k: the accumulated tensor applied to the target's moment once
        const float2 m2 = ff_dup(-2.0f);
        const float2 gx = __ffma2_rn(sq.gxz, tg.uz, __ffma2_rn(sq.gxy, tg.uy, __fmul2_rn(sq.gxx, tg.ux)));
        const float2 gy = __ffma2_rn(sq.gyz, tg.uz, __ffma2_rn(sq.gyy, tg.uy, __fmul2_rn(sq.gxy, tg.ux)));
        const float2 gz = __ffma2_rn(sq.gzz, tg.uz, __ffma2_rn(sq.gyz, tg.uy, __fmul2_rn(sq.gxz, tg.ux)));
        s.fx = __ffma2_rn(m2, gx, s.fx); s.fy = __ffma2_rn(m2, gy, s.fy); s.fz = __ffma2_rn(m2, gz, s.fz);
    }
    if (!QUAD) {
        // f_k = G u_k (Eq. 12 is linear in u_k); the result goes where the vector form keeps it
        ff_accg2_apply(sg, tg.ux, tg.uy, tg.uz, s.fx, s.fy, s.fz);
        s.hx = sg.hx; s.hy = sg.hy; s.hz = sg.hz;
        s.sk = ff_dup(0.0f);
    }
    // (the moments are read back from the packed target registers: keeping the loaded float4 alive across the
    // walk makes ptxas rebuild the register pairs with MOVs inside the evaluation loop)
    auto store = [&](int k, float ux, float uy, float uz, float hx, float hy, float hz, float fvx, float fvy, float fvz,
                     float sk) {
        FF_CHECK(g, k >= 0 && k < n && __ldg(perm + k) < (uint32_t)n);
        const size_t o = (size_t)__ldg(perm + k) * 3;      // a7: back to caller order;  f = fv + sk u_k
        if (H_out) { H_out[o] = hx; H_out[o + 1] = hy; H_out[o + 2] = hz; }
        if (F_out) { F_out[o] = fmaf(sk, ux, fvx); F_out[o + 1] = fmaf(sk, uy, fvy); F_out[o + 2] = fmaf(sk, uz, fvz); }
    };
    if (W == 32) {
        if ((half ? i1 : i0) < nm) {
            if (half) store(k1, tg.ux.y, tg.uy.y, tg.uz.y, s.hx.y, s.hy.y, s.hz.y, s.fx.y, s.fy.y, s.fz.y, s.sk.y);
            else store(k0, tg.ux.x, tg.uy.x, tg.uz.x, s.hx.x, s.hy.x, s.hz.x, s.fx.x, s.fy.x, s.fz.x, s.sk.x);
        }
    } else {
        if (i0 < nm) store(k0, tg.ux.x, tg.uy.x, tg.uz.x, s.hx.x, s.hy.x, s.hz.x, s.fx.x, s.fy.x, s.fz.x, s.sk.x);
        if (i1 < nm) store(k1, tg.ux.y, tg.uy.y, tg.uz.y, s.hx.y, s.hy.y, s.hz.y, s.fx.y, s.fy.y, s.fz.y, s.sk.y);
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
template <int W, bool COUNT, bool BUCKET, bool QUAD>
__global__ void __launch_bounds__(FF_WALK_WARPS * 32, QUAD ? FF_WALK_MINB_QUAD : FF_WALK_MINB)
ff_k_walk(int n, int group_begin, int group_end, float theta, ff_globals* __restrict__ g, const float4* __restrict__ pos_s,
          const float4* __restrict__ mom_s, const uint32_t* __restrict__ perm,
          const int4* __restrict__ cell_info, const int4* __restrict__ cell_child,
          const int32_t* __restrict__ leaf_count, const float4* __restrict__ centre,
          const float4* __restrict__ moment, const float4* __restrict__ quad, float* __restrict__ H_out,
          float* __restrict__ F_out, unsigned long long* __restrict__ counters)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    ff_walk_smem<W, QUAD>& sm = reinterpret_cast<ff_walk_smem<W, QUAD>*>(smem_raw)[w];
    const int groups = group_end;                          // groups [group_begin, group_end) of the sorted order
    const int n_cells = g->n_cells;
    for (;;) {
        int grp = 0;
        if (lane == 0) grp = group_begin + atomicAdd(&g->walk_next, 1);
        grp = __shfl_sync(FF_FULL, grp, 0);
        if (grp >= groups) break;
        ff_walk_group<W, COUNT, BUCKET, QUAD>(sm, grp, lane, n, theta, n_cells, pos_s, mom_s, perm, cell_info, cell_child,
                                              leaf_count, centre, moment, quad, H_out, F_out, counters, g);
        __syncwarp();
    }
}

template <int W, bool COUNT, bool BUCKET, bool QUAD>
static int ff_launch_walk_t(ff_ctx* c, float* H_out, float* F_out, int group_begin, int group_end, int variant)
{
    const int n = (int)c->n;
    const int groups = group_end - group_begin;
    const size_t smem = sizeof(ff_walk_smem<W, QUAD>) * FF_WALK_WARPS;
    int& per_sm = c->occ_walk[variant];                    // per context: contexts may live on different devices
    if (!per_sm) {
        FF_CUDA(c, cudaFuncSetAttribute(ff_k_walk<W, COUNT, BUCKET, QUAD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        FF_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ff_k_walk<W, COUNT, BUCKET, QUAD>, FF_WALK_WARPS * 32, smem));
        if (per_sm < 1) return FF_ERR_CUDA;
    }
    const int blocks = min(c->num_sms * per_sm, (groups + FF_WALK_WARPS - 1) / FF_WALK_WARPS);
    if (COUNT) FF_CUDA(c, cudaMemsetAsync(c->g->counters, 0, sizeof(c->g->counters), c->stream));
    auto kernel = ff_k_walk<W, COUNT, BUCKET, QUAD>;
    FF_LAUNCH(c, kernel, blocks, FF_WALK_WARPS * 32, smem, n, group_begin, group_end, c->theta, c->g,
              c->pos_s, c->mom_s, c->idx[0], c->cell_info, (const int4*)c->cell_child, c->leaf_count, c->cell_centre,
              c->cell_moment, c->cell_quad, H_out, F_out, c->g->counters);
    return FF_OK;
}

int ff_launch_walk(ff_ctx* c, float* H_out, float* F_out, int group_begin, int group_end)
{
    const int n = (int)c->n, W = c->group;
    if (group_end < 0) group_end = (n + W - 1) / W;
    if (group_end - group_begin <= 0) return FF_OK;
    const int cnt = c->count_enabled ? 1 : 0, bucket = c->nleaf > 1 ? 1 : 0;
    const int variant = (W == 64 ? 4 : (c->order == 1 ? 8 : 0)) + 2 * cnt + bucket;
    switch (variant) {
    case 0: return ff_launch_walk_t<32, false, false, false>(c, H_out, F_out, group_begin, group_end, variant);
    case 1: return ff_launch_walk_t<32, false, true, false>(c, H_out, F_out, group_begin, group_end, variant);
    case 2: return ff_launch_walk_t<32, true, false, false>(c, H_out, F_out, group_begin, group_end, variant);
    case 3: return ff_launch_walk_t<32, true, true, false>(c, H_out, F_out, group_begin, group_end, variant);
    case 4: return ff_launch_walk_t<64, false, false, false>(c, H_out, F_out, group_begin, group_end, variant);
    case 5: return ff_launch_walk_t<64, false, true, false>(c, H_out, F_out, group_begin, group_end, variant);
    case 6: return ff_launch_walk_t<64, true, false, false>(c, H_out, F_out, group_begin, group_end, variant);
    case 7: return ff_launch_walk_t<64, true, true, false>(c, H_out, F_out, group_begin, group_end, variant);
    case 8: return ff_launch_walk_t<32, false, false, true>(c, H_out, F_out, group_begin, group_end, variant);
    case 9: return ff_launch_walk_t<32, false, true, true>(c, H_out, F_out, group_begin, group_end, variant);
    case 10: return ff_launch_walk_t<32, true, false, true>(c, H_out, F_out, group_begin, group_end, variant);
    default: return ff_launch_walk_t<32, true, true, true>(c, H_out, F_out, group_begin, group_end, variant);
    }
}
