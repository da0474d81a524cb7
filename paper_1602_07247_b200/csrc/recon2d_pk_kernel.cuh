// recon2d_pk_kernel.cuh -- kernel body of recon2d_pk.cuh (which documents layout and packing).
#pragma once

namespace ants {

// METHOD 0 Poisson ML, 1 weighted chi-square.  Requires every LRF strictly positive (host-checked).
// REUSE: carry the scores of coinciding nodes over from the previous grid (see "Node reuse" below).
// LOCKSTEP: the CTA takes its events in rounds of one event per warp behind a barrier (see "Event distribution" below).
// The host picks both (make_plan in ants_recon.cu; measured per workload in profiles/r02_lockstep.md): reuse whenever
// the contraction factor is 1/2 and G is odd, with the rounds except for Poisson ML on large arrays.
template <int NPT, int METHOD, bool REUSE, bool LOCKSTEP = false>
__global__ void __launch_bounds__(256, (NPT <= 3 ? 3 : 2)) recon2d_pk_kernel(const Params p) {
    extern __shared__ __align__(16) unsigned char smem[];
    const ModelDev &m = p.m;
    const int N = m.N, nr1 = m.n_r + 1;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int rows = m.n_lrf * nr1;

    // ---- CTA-shared tables ----
    float4 *sens_s = reinterpret_cast<float4 *>(smem);
    float4 *poly_s = sens_s + N;
    int *grp_s = reinterpret_cast<int *>(poly_s + rows);
    for (int i = threadIdx.x; i < N; i += blockDim.x) { sens_s[i] = m.sens[i]; grp_s[i] = m.grp[i]; }
    for (int i = threadIdx.x; i < rows; i += blockDim.x) poly_s[i] = m.poly[i];
    float2 *node_s = reinterpret_cast<float2 *>(smem + cta_table_bytes(N, rows));
    constexpr int slots = 32 * NPT;
    {
        const float halfg = 0.5f * (float)(p.G - 1);
        for (int n = threadIdx.x; n < slots; n += blockDim.x) {
            const int iy = n / p.G, ix = n - iy * p.G;
            node_s[n] = n < p.nodes ? make_float2((float)ix - halfg, (float)iy - halfg) : make_float2(0.f, 0.f);
        }
    }
    // Node reuse, static part: with a previous winner far enough from the border of its grid, the nodes that coincide
    // with old ones (both offsets from the centre even) and the ones to evaluate are the same lists in every
    // iteration; only a winner near the border needs the lists built for it.
    unsigned char *ident_s = reinterpret_cast<unsigned char *>(node_s + slots);     // 0, 1, 2, ...: every node
    unsigned char *todo_s = ident_s + slots, *even_s = todo_s + slots;
    short *evoff_s = reinterpret_cast<short *>(even_s + slots);
    int *lists_s = reinterpret_cast<int *>(evoff_s + slots);         // {n_todo, n_even, reach of the even offsets}
    if (REUSE)
        for (int n = threadIdx.x; n < slots; n += blockDim.x) ident_s[n] = (unsigned char)n;
    if (REUSE && warp == 0) {
        const int hg = (p.G - 1) >> 1;
        const unsigned ltm = (1u << lane) - 1u;
        int ct = 0, ce = 0, mr = 0;
        for (int n0 = 0; n0 < p.nodes; n0 += 32) {
            const int n = n0 + lane, iy = n / p.G, ix = n - iy * p.G, dxn = ix - hg, dyn = iy - hg;
            const bool valid = n < p.nodes, even = valid && !((dxn | dyn) & 1);
            const unsigned mt = __ballot_sync(kFull, valid && !even), me = __ballot_sync(kFull, even);
            if (valid && !even) todo_s[ct + __popc(mt & ltm)] = (unsigned char)n;
            if (even) {
                const int q = ce + __popc(me & ltm);
                even_s[q] = (unsigned char)n;
                evoff_s[q] = (short)((dyn >> 1) * p.G + (dxn >> 1));
                mr = max(mr, max(abs(dxn >> 1), abs(dyn >> 1)));
            }
            ct += __popc(mt);
            ce += __popc(me);
        }
        mr = __reduce_max_sync(kFull, mr);
        if (lane == 0) { lists_s[0] = ct; lists_s[1] = ce; lists_s[2] = mr; }
    }
    __syncthreads();
    WarpSmemPk w = carve_pk(smem + (cta_smem_bytes_pk(N, rows, NPT) + 15) / 16 * 16 +
                            (size_t)warp * warp_smem_bytes_pk(N, METHOD, p.nodes), N, METHOD, p.nodes);
    const int np1 = pk_pairs(N);
    const unsigned poly_base = (unsigned)__cvta_generic_to_shared(poly_s) - ((unsigned)kMagicBits << 4);

    // this lane's nodes: offsets from the grid centre in units of the step
    const float half = 0.5f * (float)(p.G - 1);
    const float half_diag_units = 1.41421356f * half;
    const f32x2 sc2 = pk1(m.sc), of2 = pk1(m.of), magic2 = pk1(kMagic), nmagic2 = pk1(-kMagic);

    // The next event's signals are fetched while this one runs: into registers (4 per lane: N <= 128) in the
    // instantiations with up to three nodes per lane, into L2 only (prefetch.global.L2) in the larger ones, where four
    // more registers held across the search cost the node loops their in-place accumulators (register copies at every
    // loop back-edge of the chi-square node-reuse kernel).
    constexpr bool kRegPrefetch = NPT <= 3;
    float pf[4];
    auto prefetch = [&](long long ev) {
        if (kRegPrefetch) {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const int i = lane + 32 * c;
                pf[c] = (ev < p.n_events && i < N) ? __ldg(p.signals + ev * N + i) : 0.f;
            }
        } else if (ev < p.n_events) {
            for (int i = lane * 32; i < N; i += 32 * 32)       // one request per 128-byte line of the row
                asm volatile("prefetch.global.L2 [%0];" ::"l"(p.signals + ev * N + i));
        }
    };
    // Event distribution.  Default: every warp takes its next event from the launch's counter on its own.  LOCKSTEP:
    // the CTA takes `warps` consecutive events per round behind a barrier, so its warps walk through the phases of
    // the search together and share the instruction caches: the kernel's code is several times their size, and the
    // node-reuse instantiations, with two sets of node loops, stalled on instruction fetch 1.9 warps per issue slot on
    // config 3 (0.4 without reuse).  It pays where the events of a CTA take about the same time (profiles/r02_lockstep.md).
    __shared__ long long round_s;
    const int warps = blockDim.x >> 5;
    long long b_next = LOCKSTEP ? grab_round(p.ctr, warps, &round_s) : 0;
    long long e_next = LOCKSTEP ? b_next + warp : grab_event(p.ctr, lane);
    prefetch(e_next);
    for (long long e = e_next; LOCKSTEP ? b_next < p.n_events : e < p.n_events; e = e_next) {
        if (LOCKSTEP) {
            b_next = grab_round(p.ctr, warps, &round_s);
            e_next = b_next + warp;
            if (e >= p.n_events) continue;       // (the last round may be short)
        } else {
            e_next = grab_event(p.ctr, lane);
        }
        // ---- a1: signals (requested into L2 while the previous event ran), centroid / strongest-sensor start,
        // selection (prepare_event, recon_common.cuh); the next event's row is requested before this one is searched
        float cur[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) cur[c] = kRegPrefetch ? pf[c] : 0.f;
        prefetch(e_next);
        float sumS, cx, cy;
        if (!prepare_event<METHOD>(p, sens_s, w.SC, e, lane, sumS, cx, cy, kRegPrefetch ? cur : nullptr)) continue;

        // reference energy for the plain score: A at the seed
        float A_ref;
        {
            float sl = 0.f;
            for (int i = lane; i < N; i += 32) {
                float4 sn = sens_s[i];
                float dx = cx - sn.x, dy = cy - sn.y;
                float s = eval_axial(m, poly_s + grp_s[i] * nr1, sqrt_approx(fmaf(dx, dx, dy * dy)));
                if (w.SC[i].y == w.SC[i].y) sl += sn.z * s;
            }
            sl = warp_sum(sl);
            A_ref = sl > 0.f ? sumS * rcp_approx(sl) : 1.f;   // only conditions the plain score
        }

        // Node reuse.  With a contraction of 1/2 and an odd G the nodes of the new grid that sit an even number of
        // steps from its centre coincide with nodes of the previous grid (25 of 81, 25 of 121): their scores are
        // carried over -- a plain score as it is, a differential one minus the new centre's -- and only the other
        // nodes are evaluated, compacted onto the lanes (9 x 9: two rounds of 32 instead of three).  Not across the
        // switch from the plain to the differential score, nor after an iteration without a valid node.
        const bool reuse_ok = REUSE && p.factor == 0.5f && (p.G & 1);
        float *sc_prev = w.S0, *sc_cur = w.S1;
        bool have_prev = false;
        int prev_bi = 0, prev_bx = 0, prev_by = 0, prev_mode = -1;
        const unsigned lt = (1u << lane) - 1u;

        float h = p.h0_xy;
        for (int k = 0; k < p.K; ++k) {
            const int mode = k < p.k_diff ? 0 : 1;
            // ---- the nodes of this iteration: carried over or to be evaluated ----
            int count = p.nodes;
            const unsigned char *lst = ident_s;
            if (REUSE && reuse_ok && have_prev && mode == prev_mode) {
                const float off = mode == 1 ? sc_prev[prev_bi] : 0.f;
                const int mr = lists_s[2];
                if (prev_bx >= mr && prev_bx + mr < p.G && prev_by >= mr && prev_by + mr < p.G) {
                    // every coinciding node lies inside the previous grid: the static lists
                    const int n_even = lists_s[1];
                    for (int t = lane; t < n_even; t += 32) sc_cur[even_s[t]] = sc_prev[prev_bi + evoff_s[t]] - off;
                    count = lists_s[0];
                    lst = todo_s;
                } else {
                    count = 0;
#pragma unroll
                    for (int j = 0; j < NPT; ++j) {
                        const int n = lane + 32 * j;
                        bool todo = n < p.nodes;
                        if (todo) {
                            const float2 no = node_s[n];
                            const int dxn = (int)no.x, dyn = (int)no.y;      // steps from the centre (G odd: integers)
                            const int ox = prev_bx + (dxn >> 1), oy = prev_by + (dyn >> 1);
                            if (!((dxn | dyn) & 1) && (unsigned)ox < (unsigned)p.G && (unsigned)oy < (unsigned)p.G) {
                                sc_cur[n] = sc_prev[oy * p.G + ox] - off;
                                todo = false;
                            }
                        }
                        const unsigned mk = __ballot_sync(kFull, todo);
                        if (todo) w.L[count + __popc(mk & lt)] = (unsigned char)n;
                        count += __popc(mk);
                    }
                    __syncwarp();
                    lst = w.L;
                }
            }
            int nid[NPT];
#pragma unroll
            for (int j = 0; j < NPT; ++j)
                nid[j] = !REUSE ? lane + 32 * j : lane + 32 * j < count ? (int)lst[lane + 32 * j] : 0;

            float sc_node[NPT];          // scores of this lane's nodes (lower is better), +inf = invalid
            float aux_node[NPT];         // plain mode: sum L (Poisson) / A (chi2) at the node
            // (the sensor-pair loops inside are compiled for NPT and for NPT - 1 nodes per lane, statically unrolled:
            // the shorter ones serve when the carried-over nodes free a whole round of 32 lanes)
            const bool short_round = REUSE && NPT > 1 && count <= 32 * (NPT - 1);
            if (mode == 0) {
#include "recon2d_pk_plain.inc"
            } else {
#include "recon2d_pk_diff.inc"
            }
            if (REUSE) {
#pragma unroll
                for (int j = 0; j < NPT; ++j)     // (four nodes per lane: the ids are read again rather than kept across
                                                  // the node loops, whose accumulators need the registers)
                    if (lane + 32 * j < count) sc_cur[NPT >= 4 ? (int)lst[lane + 32 * j] : nid[j]] = sc_node[j];
                __syncwarp();
            }

            // ---- a5: argmin over the G^2 nodes in their natural order (R9), recentre, contract ----
            float bs = kInf;
            int bi = 0x7fffffff;
#pragma unroll
            for (int j = 0; j < NPT; ++j) {
                const int n = lane + 32 * j;
                const float sv = !REUSE ? sc_node[j] : n < p.nodes ? sc_cur[n] : kInf;
                if (sv < bs) { bs = sv; bi = n; }
            }
            warp_argmin_redux(bs, bi);
            const bool found = bs < kInf;
            if (found) {
                if (mode == 0 && !REUSE) {
                    // (with node reuse the reference energy stays at its seed value: the plain score's rounding
                    // error depends on it, alike for all nodes of one grid but not from one grid to the next, and
                    // carried-over scores are compared with fresh ones)
                    // the winner's energy, if it was evaluated in this iteration, lives in the lane that scored it
                    float mine = 0.f;
                    bool has = false;
#pragma unroll
                    for (int j = 0; j < NPT; ++j)
                        if (lane + 32 * j < count && nid[j] == bi) { mine = aux_node[j]; has = true; }
                    const unsigned who = __ballot_sync(kFull, has);
                    if (who) {
                        const float v = __shfl_sync(kFull, mine, __ffs(who) - 1);
                        A_ref = METHOD == 0 ? sumS * rcp_approx(v) : v;
                    }
                }
                const float2 wo = node_s[bi];           // the winner's grid offsets (one broadcast load)
                cx = fmaf(wo.x, h, cx);
                cy = fmaf(wo.y, h, cy);
                if (REUSE) {                            // its column and row (G odd: the offsets are integers)
                    prev_bx = (int)wo.x + ((p.G - 1) >> 1);
                    prev_by = (int)wo.y + ((p.G - 1) >> 1);
                }
            }
            if (p.out_path && lane == 0) p.out_path[e * p.K + k] = found ? (uint16_t)bi : (uint16_t)0xFFFF;
            h *= p.factor;
            have_prev = found;
            prev_bi = found ? bi : 0;
            prev_mode = mode;
            float *tmp = sc_prev;
            sc_prev = sc_cur;
            sc_cur = tmp;
            __syncwarp();
        }

        // ---- a6: FP64 energy and score at the final node, store ----
        float A_fin, score_fin;
        WarpSmem2D w2;               // final_score_2d needs N doubles of scratch (D[0..1]) and SC
        w2.A = w.D[0];
        w2.SC = w.SC;
        final_score_2d<METHOD>(m, sens_s, grp_s, w2, lane, cx, cy, A_fin, score_fin);
        if (lane == 0) {
            reinterpret_cast<float4 *>(p.out_xyzA)[e] = make_float4(cx, cy, 0.f, A_fin);
            p.out_score[e] = score_fin;
        }
    }
    retire_warp(p.ctr, p.total_warps, lane);
}

}  // namespace ants
