// recon2d_pk_kernel.cuh -- kernel body of recon2d_pk.cuh (which documents layout and packing).
#pragma once

namespace ants {

// METHOD 0 Poisson ML, 1 weighted chi-square.  Requires every LRF strictly positive (host-checked).
template <int NPT, int METHOD>
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
    {
        const float halfg = 0.5f * (float)(p.G - 1);
        for (int n = threadIdx.x; n < 256; n += blockDim.x) {
            const int iy = n / p.G, ix = n - iy * p.G;
            node_s[n] = n < p.nodes ? make_float2((float)ix - halfg, (float)iy - halfg) : make_float2(0.f, 0.f);
        }
    }
    __syncthreads();
    WarpSmemPk w = carve_pk(smem + (cta_smem_bytes_pk(N, rows) + 15) / 16 * 16 +
                            (size_t)warp * warp_smem_bytes_pk(N, METHOD), N, METHOD);
    const int np1 = pk_pairs(N);
    const unsigned poly_base = (unsigned)__cvta_generic_to_shared(poly_s) - ((unsigned)kMagicBits << 4);

    // this lane's nodes: offsets from the grid centre in units of the step
    const float half = 0.5f * (float)(p.G - 1);
    const float half_diag_units = 1.41421356f * half;
    const f32x2 sc2 = pk1(m.sc), of2 = pk1(m.of), magic2 = pk1(kMagic), nmagic2 = pk1(-kMagic);

    // the next event's signals are fetched into registers (4 per lane: N <= 128) while this one runs
    float pf[4];
    auto prefetch = [&](long long ev) {
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const int i = lane + 32 * c;
            pf[c] = (ev < p.n_events && i < N) ? __ldg(p.signals + ev * N + i) : 0.f;
        }
    };
    long long e_next = grab_event(p.ctr, lane);
    prefetch(e_next);
    for (long long e = e_next; e < p.n_events; e = e_next) {
        e_next = grab_event(p.ctr, lane);
        // ---- a1: signals (prefetched while the previous event ran), centroid / strongest-sensor start, selection
        // (prepare_event, recon_common.cuh); the next event's row is requested before this one is searched
        float cur[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) cur[c] = pf[c];
        prefetch(e_next);
        float sumS, cx, cy;
        if (!prepare_event<METHOD>(p, sens_s, w.SC, e, lane, sumS, cx, cy, cur)) continue;

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

        float h = p.h0_xy;
        for (int k = 0; k < p.K; ++k) {
            float sc_node[NPT];          // node scores (lower is better), +inf = invalid
            float aux_node[NPT];         // plain mode: sum L (Poisson) / A (chi2) at the node
            if (k < p.k_diff) {
#include "recon2d_pk_plain.inc"
            } else {
#include "recon2d_pk_diff.inc"
            }

            // ---- a5: argmin over the G^2 nodes, recentre, contract ----
            float bs = kInf;
            int bi = 0x7fffffff;
#pragma unroll
            for (int j = 0; j < NPT; ++j)
                if (sc_node[j] < bs) { bs = sc_node[j]; bi = lane + 32 * j; }
            warp_argmin_redux(bs, bi);
            const bool found = bs < kInf;
            if (found) {
                if (k < p.k_diff) {
                    float mine = 0.f;
#pragma unroll
                    for (int j = 0; j < NPT; ++j)
                        if ((bi >> 5) == j) mine = aux_node[j];
                    float v = __shfl_sync(kFull, mine, bi & 31);
                    A_ref = METHOD == 0 ? sumS * rcp_approx(v) : v;
                }
                const float2 wo = node_s[bi];           // the winner's grid offsets (one broadcast load)
                cx = fmaf(wo.x, h, cx);
                cy = fmaf(wo.y, h, cy);
            }
            if (p.out_path && lane == 0) p.out_path[e * p.K + k] = found ? (uint16_t)bi : (uint16_t)0xFFFF;
            h *= p.factor;
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
