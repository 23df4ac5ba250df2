// fstat_fastmulti.cu -- row f4 (Eq. 3; A, E, T of PAPER.md:48, reading A28): the interpolating kernel for
// two or three TDI channels of the A / E / T family in ONE pass.  What the channels share is evaluated once:
//   * per node: the SPA phase, t_f, the orbit, the three arms seen from both ends and the Michelson responses
//     X', Y', Z' (michelson_xyz); a channel is three weights on them;
//   * per bin: the carrier e^{+i Phi} (rotation recurrence, 9 FP64 instructions) -- the phase is the same for every
//     channel of a template; each channel adds its own q = dw'_ch E and running sums A_0..A_3 (10 instructions).
// Per bin 9 + 10 n_ch FP64 instructions against 19 n_ch for one pass per channel.  Each channel keeps its own data
// stream (TMA tiles), Gram tables (its own noise weights) and eight sums, written to its own plan's partial-sum
// array in the layout of fstat_fast_kernel, so that the direct kernel and the epilogue are unchanged.
// CTA = 128 threads = 128 particles, 2 CTAs per SM (node ring 1 + 4 n_ch values x 6 nodes per thread in shared
// memory, 256-bin tiles in two stages).  Product path only.
#include "fstat_fast.cuh"
#include "fstat_model.cuh"

namespace fstat {

constexpr int kMTileShift = 8;
constexpr int kMTile = 1 << kMTileShift;      // bins per tile and channel (4 KiB); a 512-bin node interval spans two
constexpr int kMStages = 2;

template <int NCH>
struct __align__(16) MultiSmem {
    double2 tile[kMStages][NCH][kMTile];
    double win[kWinNodes][1 + 4 * NCH][kThreads];
    uint64_t full[kMStages];
};

template <int NCH>
__global__ void __launch_bounds__(kThreads, 2) fstat_fastmulti_kernel(const __grid_constant__ FastMultiArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    MultiSmem<NCH> &sm = *reinterpret_cast<MultiSmem<NCH> *>(smem_raw);

    const int tid = threadIdx.x;
    const int grp = blockIdx.x % a.n_groups;
    const int chunk = blockIdx.x / a.n_groups;
    const int seg_begin = chunk * a.segs_per_cta, seg_end = min(a.n_seg, seg_begin + a.segs_per_cta);
    const int8_t *level = a.level + (int64_t)grp * a.n_seg;
    const int64_t p = (int64_t)grp * kThreads + tid;         // < P_pad by construction
    const double *cf = a.coef + p;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < kMStages; ++s) mbar_init(&sm.full[s], 1);
        mbar_fence_init();
    }
    __syncthreads();
    int g0 = 0;                                              // tiles consumed so far by this CTA (ring position)

  for (int seg = seg_begin; seg < seg_end;) {
    const int lvl = level[seg];
    if (lvl < 0) { ++seg; continue; }                        // CTA-uniform
    int run_end = seg + 1;
    while (run_end < seg_end && level[run_end] == lvl) ++run_end;
    const int sh = kLevel0Shift + lvl;
    const double rS = 1.0 / (double)(1 << sh);

    const int lo = a.seg_edge[seg], hi = a.seg_edge[run_end];
    const int t_first = lo >> kMTileShift;
    const int n_tiles = ((hi - 1) >> kMTileShift) - t_first + 1;

    auto issue_tile = [&](int t) {                           // t = tile number relative to t_first
        const int slot = (g0 + t) % kMStages;
        const int b0 = max(lo, (t_first + t) << kMTileShift), b1 = min(hi, (t_first + t + 1) << kMTileShift);
        const uint32_t bytes = (uint32_t)(b1 - b0) * (uint32_t)sizeof(double2);
        mbar_expect_tx(&sm.full[slot], bytes * NCH);
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch)
            tma_load_1d(&sm.tile[slot][ch][b0 & (kMTile - 1)], reinterpret_cast<const double2 *>(a.dwp[ch]) + b0, bytes,
                        &sm.full[slot]);
    };
    __syncthreads();                                         // every thread has left the previous run's tiles
    if (tid == 0)
        for (int s = 0; s < kMStages && s < n_tiles; ++s) issue_tile(s);

    const double c0 = cf[0];
    const double slope = mulmod4(c0, a.df);

    // node ring: psi_nl, then (T'_+ re, im, T'_x re, im) of every channel, at the last six nodes
    auto eval_node = [&](int mnode) {
        double c[kNCoef];
        load_coef(cf, a.P_pad, c);
        const double2 *row = reinterpret_cast<const double2 *>(
            a.node + ((int64_t)kNodePad + ((int64_t)mnode * (1 << lvl))) * kTabW);
        NodeGeom g;
        node_geometry(row, c, a.orb, g);
        double xyz[2][6];
        michelson_xyz(g, xyz);
        const int slot = (mnode + kWinNodes) % kWinNodes;
        sm.win[slot][0][tid] = g.psi_nl;
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
            const double wx = a.wch[ch][0], wy = a.wch[ch][1], wz = a.wch[ch][2];
#pragma unroll
            for (int pol = 0; pol < 2; ++pol) {
                sm.win[slot][1 + 4 * ch + 2 * pol][tid] = fma(wx, xyz[pol][0], fma(wy, xyz[pol][2], wz * xyz[pol][4]));
                sm.win[slot][2 + 4 * ch + 2 * pol][tid] = fma(wx, xyz[pol][1], fma(wy, xyz[pol][3], wz * xyz[pol][5]));
            }
        }
    };
    int m = lo >> sh;
    for (int k = -2; k <= 2; ++k) eval_node(m + k);
    int m_have = m + 2;                                      // highest node in the ring

    double acc[NCH][kNAcc];
    double c_re[NCH], c_im[NCH];
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
#pragma unroll
        for (int j = 0; j < kNAcc; ++j) acc[ch][j] = 0.0;
        c_re[ch] = c_im[ch] = 0.0;
    }

    int64_t gidx = (int64_t)a.seg_gbase[seg * kNLevels + lvl] * kNW;
    int cur_tile = -1;
    int cur_seg = seg;
    int seg_hi = a.seg_edge[cur_seg + 1];
    bool seg_start = true;                                   // basis (u_+, u_x - c u_+) chosen per segment and channel (hazard H3)
    int j0 = lo;
    while (j0 < hi) {
        const int node0 = m << sh;                           // bin of node "0" of this interval
        const int j1 = min(seg_hi, node0 + (1 << sh));       // sub-block = node interval cut at the segment edge
        const int s_base = (m - 2 + kWinNodes) % kWinNodes;  // ring slot of node m-2
        const double fnode = a.node[((int64_t)kNodePad + ((int64_t)m << lvl)) * kTabW + T_F];
        if (m + 3 > m_have) {
            m_have = m + 3;
            eval_node(m + 3);
        }
        // ---- carrier phase: economised cubic + exact linear term, as forward differences
        double t, D1, D2, D3;
        {
            double v[6], yref, e[4];
#pragma unroll
            for (int k = 0; k < 6; ++k) v[k] = sm.win[(s_base + k) % kWinNodes][0][tid];
            economise(v, yref, e);
            const double d0 = e[0] - e[1], d2 = e[2] - e[1], d3 = e[3] - e[1];
            const double a1 = fma(d0, -1.0 / 3.0, fma(d3, -1.0 / 6.0, d2));
            const double a2 = 0.5 * (d0 + d2);
            const double a3 = fma(d2, -0.5, (d3 - d0) * (1.0 / 6.0));
            const double G0 = red4(yref) + e[1] + mulmod4(c0, fnode);
            const double G1 = red4(fma(a1, rS, slope));
            const double G2 = a2 * rS * rS, G3 = a3 * rS * rS * rS;
            const double s0 = (double)(j0 - node0);
            t = fma(s0, fma(s0, fma(s0, G3, G2), G1), G0);
            D1 = fma(G3, fma(3.0 * s0, s0 + 1.0, 1.0), fma(G2, fma(2.0, s0, 1.0), G1));
            D2 = fma(G3, fma(6.0, s0, 6.0), 2.0 * G2);
            D3 = 6.0 * G3;
        }
        // ---- per bin: the carrier recurrence of fstat_fast_kernel (E <- E R, R <- R Q every bin; Q <- Q C^4 every
        // 4 bins), shared by the channels; per channel q = dw'_ch E into the running sums A_0..A_3
        double Er, Ei, Rr, Ri, Qr, Qi, Cr, Ci;
        sincos_qt(t, Ei, Er);
        sincos_qt(fma(-1.25, D3, D1), Ri, Rr);
        sincos_qt_small(fma(1.5, D3, D2), Qi, Qr);
        sincos_qt_small(4.0 * D3, Ci, Cr);
        double A[NCH][8];
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch)
#pragma unroll
            for (int j = 0; j < 8; ++j) A[ch][j] = 0.0;
#define FSTAT_CH_STEP(ch, d)                                                                         \
        {                                                                                            \
            A[ch][0] = fma((d).x, Er, fma(-(d).y, Ei, A[ch][0]));                                    \
            A[ch][1] = fma((d).x, Ei, fma((d).y, Er, A[ch][1]));                                     \
            A[ch][2] += A[ch][0]; A[ch][3] += A[ch][1];                                              \
            A[ch][4] += A[ch][2]; A[ch][5] += A[ch][3];                                              \
            A[ch][6] += A[ch][4]; A[ch][7] += A[ch][5];                                              \
        }
#define FSTAT_CARRIER_STEP()                                                                         \
        {                                                                                            \
            const double er = fma(Er, Rr, -Ei * Ri);                                                 \
            Ei = fma(Er, Ri, Ei * Rr);                                                               \
            Er = er;                                                                                 \
            const double rr = fma(Rr, Qr, -Ri * Qi);                                                 \
            Ri = fma(Rr, Qi, Ri * Qr);                                                               \
            Rr = rr;                                                                                 \
        }
        // the 4-bin runs of the recurrence are counted from j0 across the tile boundaries inside the sub-block
        int jj = j0;
        int phase4 = 0;                                      // bins done since the last Q update
        while (jj < j1) {
            const int tl = (jj >> kMTileShift) - t_first;
            if (tl != cur_tile) {
                if (cur_tile >= 0) {
                    __syncthreads();                         // every thread is done with the previous tile
                    if (tid == 0 && cur_tile + kMStages < n_tiles) issue_tile(cur_tile + kMStages);
                }
                cur_tile = tl;
                mbar_wait(&sm.full[(g0 + tl) % kMStages], (uint32_t)(((g0 + tl) / kMStages) & 1));
            }
            const int pe = min(j1, (t_first + tl + 1) << kMTileShift);      // end of the piece inside this tile
            const int st = (g0 + tl) % kMStages;
            const int off = jj & (kMTile - 1);
            const int nb = pe - jj;
            int b = 0;
            while (b < nb) {
                if (phase4 == 0 && b + 4 <= nb) {
                    for (; b + 4 <= nb; b += 4) {
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
#pragma unroll
                            for (int ch = 0; ch < NCH; ++ch) {
                                const double2 d = sm.tile[st][ch][off + b + u];
                                FSTAT_CH_STEP(ch, d)
                            }
                            FSTAT_CARRIER_STEP()
                        }
                        const double qq = fma(Qr, Cr, -Qi * Ci);
                        Qi = fma(Qr, Ci, Qi * Cr);
                        Qr = qq;
                    }
                    continue;
                }
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch) {
                    const double2 d = sm.tile[st][ch][off + b];
                    FSTAT_CH_STEP(ch, d)
                }
                FSTAT_CARRIER_STEP()
                ++b;
                if (++phase4 == 4) {
                    phase4 = 0;
                    const double qq = fma(Qr, Cr, -Qi * Ci);
                    Qi = fma(Qr, Ci, Qi * Cr);
                    Qr = qq;
                }
            }
            jj = pe;
        }
#undef FSTAT_CH_STEP
#undef FSTAT_CARRIER_STEP

        const double U = (double)(j1 - node0);
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
            // ---- the slow factors of this interval and channel: node values at t = -2 .. 3
            double vpr[6], vpi[6], vcr[6], vci[6];
#pragma unroll
            for (int k = 0; k < 6; ++k) {
                const int sl = (s_base + k) % kWinNodes;
                vpr[k] = sm.win[sl][1 + 4 * ch][tid]; vpi[k] = sm.win[sl][2 + 4 * ch][tid];
                vcr[k] = sm.win[sl][3 + 4 * ch][tid]; vci[k] = sm.win[sl][4 + 4 * ch][tid];
            }
            if (seg_start) {
                const double n2 = fma(vpr[2], vpr[2], vpi[2] * vpi[2]), x2 = fma(vcr[2], vcr[2], vci[2] * vci[2]);
                const bool use = n2 > 1e-6 * x2;                              // else T'_+ ~ 0 there: keep u_x
                const double inv = use ? 1.0 / n2 : 0.0;
                c_re[ch] = fma(vcr[2], vpr[2], vci[2] * vpi[2]) * inv;       // T'_x conj(T'_+) / |T'_+|^2 at node "0"
                c_im[ch] = fma(vci[2], vpr[2], -vcr[2] * vpi[2]) * inv;
            }
#pragma unroll
            for (int k = 0; k < 6; ++k) {                                    // node values of T'_x - c T'_+
                vcr[k] -= fma(c_re[ch], vpr[k], -c_im[ch] * vpi[k]);
                vci[k] -= fma(c_re[ch], vpi[k], c_im[ch] * vpr[k]);
            }
            // ---- z_P += sum_k conj(v^P_k) B_k
            {
                double Br[6], Bi[6];
                subblock_weights(A[ch], rS, U, Br, Bi);
                z_from_nodes(vpr, vpi, Br, Bi, acc[ch][0], acc[ch][1]);
                z_from_nodes(vcr, vci, Br, Bi, acc[ch][2], acc[ch][3]);
            }
            // ---- m_PQ += (W v^P) . conj(W v^Q) with this channel's table (its own noise weights)
            {
                double mpp, mcc, mre, mim;
                gram_forms(a.gram[ch][lvl] + gidx, vpr, vpi, vcr, vci, mpp, mcc, mre, mim);
                acc[ch][4] += mpp; acc[ch][5] += mcc; acc[ch][6] += mre; acc[ch][7] += mim;
            }
        }
        seg_start = false;
        gidx += kNW;
        if (j1 == seg_hi) {                                  // segment finished: flush the eight sums of every channel
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch) {
                double *out = a.partial[ch] + ((int64_t)cur_seg * kNPartial) * a.P_pad + p * a.part_sp;
#pragma unroll
                for (int j = 0; j < kNAcc; ++j) { out[(int64_t)j * a.part_sk] = acc[ch][j]; acc[ch][j] = 0.0; }
                out[(int64_t)8 * a.part_sk] = c_re[ch];
                out[(int64_t)9 * a.part_sk] = c_im[ch];
            }
            seg_start = true;
            ++cur_seg;
            if (cur_seg < run_end) seg_hi = a.seg_edge[cur_seg + 1];
        }
        if (j1 == node0 + (1 << sh)) ++m;                    // node interval finished
        j0 = j1;
    }
    g0 += n_tiles;
    seg = run_end;
  }
}

cudaError_t fastmulti_kernel_configure()
{
    cudaError_t e = cudaFuncSetAttribute(fstat_fastmulti_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)sizeof(MultiSmem<2>));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(fstat_fastmulti_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)sizeof(MultiSmem<3>));
}

cudaError_t launch_fastmulti(const FastMultiArgs &a, cudaStream_t st)
{
    const int64_t n_chunks = (a.n_seg + a.segs_per_cta - 1) / a.segs_per_cta;
    const int64_t n_cta = (int64_t)a.n_groups * n_chunks;
    if (a.n_ch == 2) fstat_fastmulti_kernel<2><<<(unsigned)n_cta, kThreads, sizeof(MultiSmem<2>), st>>>(a);
    else if (a.n_ch == 3) fstat_fastmulti_kernel<3><<<(unsigned)n_cta, kThreads, sizeof(MultiSmem<3>), st>>>(a);
    else return cudaErrorInvalidValue;
    return cudaGetLastError();
}

}  // namespace fstat
