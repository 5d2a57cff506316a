// giant_resident.cuh -- giant steps (Eq. 4, or its Clenshaw form, reading A6) for
// small N (N <= 512), as ONE persistent launch in which
//   * every CTA keeps its 32-row block of the multiplier Y = T_k resident in shared memory for all p-1
//     products (the A operand never changes along the chain: 32 x Kpad x 8 B <= 128 KB), so a step only
//     streams the B operand (the previous accumulator panel) from L2;
//   * every CTA runs TWO independent consumer groups (4 warps each, 32x32 output tile, own TMA ring and own
//     producer warp), one per column panel.  Column panels are independent chains (step l of panel tn needs
//     only panel tn of step l+1), so while one group sits in the latency part of its chain (store -> fence ->
//     flag -> poll -> TMA round trip) the other group's K loop owns the DMMA pipe;
//   * completion is published by the group's producer warp (mbarrier hand-off, then one gpu fence and one
//     relaxed increment), so the consumer warps go straight on to the prologue of their next step.
// This replaces, for the serial part of the solve, the stream-level concurrency of PAPER.md:228-232 (which the
// paper found to help only below N ~ 1000): measured 13.4 -> see DESIGN.md section 6 us per giant step at N = 500.
//
// Work assignment is static: CTA b handles row block tm = b % tiles_m and the panels tn = 2 (b / tiles_m) + g,
// g = 0, 1.  All CTAs must be co-resident (cooperative launch); they synchronise only through the per-panel
// completion counters of gemm_dmma.cuh.
#pragma once
#include "gemm_dmma.cuh"

namespace chebdm {

constexpr int GR_BM = 32, GR_BN = 32, GR_BK = 32, GR_STAGES = 4;
constexpr int GR_SLAB_BYTES = GR_BK * 128;               // 4 KB: 16 columns x 32 k-rows
constexpr int GR_TILE_BYTES = 2 * GR_SLAB_BYTES;         // 8 KB: one 32-column operand block of one k-tile
constexpr int GR_GROUP_WARPS = 4;                        // 2 x 2 warps of 16 x 16
constexpr int GR_THREADS = (2 * GR_GROUP_WARPS + 2) * 32;  // two consumer groups + two producer warps
constexpr int GR_MAX_KTILES = 16;                        // N <= 512

struct GiantArgs {
    const Task* tasks;       // giant tasks: tasks[first_task + s], s = 0..nsteps-1 (s = 0 is the product-free step)
    const CUtensorMap* maps;
    int first_task, nsteps;
    int N, ktiles;
    int tiles_m, tiles_n;    // 32-row blocks, 32-column panels
    int* panel_done;         // [task][panel] completion counters (target tiles_m)
    int panel_stride;
    double* userD;
    long long ldD;
    int tma2d;
    int* error_flag;
    TraceRec* trace;         // nullable; record index = trace_base + (s * tiles_n + tn) * tiles_m + tm
    int trace_base;
};

inline int giant_resident_smem_bytes(int ktiles) {
    return ktiles * GR_TILE_BYTES + 2 * GR_STAGES * GR_TILE_BYTES + 256 + 1024;
}

__global__ void __launch_bounds__(GR_THREADS, 1) giant_resident_kernel(const GiantArgs args) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const int ktiles = args.ktiles;
    uint8_t* a_res = smem;                                        // [ktiles][8 KB]
    uint8_t* ring0 = smem + ktiles * GR_TILE_BYTES;               // [group][stage][8 KB]
    uint64_t* bars = reinterpret_cast<uint64_t*>(ring0 + 2 * GR_STAGES * GR_TILE_BYTES);
    // bars: [0] resident A; per group g: [1 + g*(2S+1) + s] full, [.. + S + s] empty, [.. + 2S] stored
    const uint32_t bar_base = smem_u32(bars);
    auto resa_bar = [&]() { return bar_base; };
    auto full_bar = [&](int g, int s) { return bar_base + 8u * (1 + g * (2 * GR_STAGES + 1) + s); };
    auto empty_bar = [&](int g, int s) { return bar_base + 8u * (1 + g * (2 * GR_STAGES + 1) + GR_STAGES + s); };
    auto stored_bar = [&](int g) { return bar_base + 8u * (1 + g * (2 * GR_STAGES + 1) + 2 * GR_STAGES); };
    auto stagger_bar = [&]() { return bar_base + 8u * (1 + 2 * (2 * GR_STAGES + 1)); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        mbar_init(resa_bar(), 1);
        for (int g = 0; g < 2; ++g) {
            for (int s = 0; s < GR_STAGES; ++s) {
                mbar_init(full_bar(g, s), 1);
                mbar_init(empty_bar(g, s), GR_GROUP_WARPS);
            }
            mbar_init(stored_bar(g), GR_GROUP_WARPS);
        }
        mbar_init(stagger_bar(), GR_GROUP_WARPS);
        fence_mbar_init();
    }
    __syncthreads();

    const int tm = blockIdx.x % args.tiles_m;
    const int pair = blockIdx.x / args.tiles_m;
    const int N = args.N;
    const int nsteps = args.nsteps;

    if (warp >= 2 * GR_GROUP_WARPS) {
        // =============================== producer warp of group g ===============================
        const int g = warp - 2 * GR_GROUP_WARPS;
        const int tn = 2 * pair + g;
        if (lane != 0) return;
        if (g == 0) {
            // resident A: rows [tm*32, tm*32+32) of Y = T_k as [k][column] blocks (Y is symmetric)
            const Task* t1 = args.tasks + args.first_task + (nsteps > 1 ? 1 : 0);
            const CUtensorMap* mapA = args.maps + t1->mapA;
            mbar_arrive_expect_tx(resa_bar(), (uint32_t)(ktiles * GR_TILE_BYTES));
            for (int kt = 0; kt < ktiles; ++kt) {
                const uint32_t dst = smem_u32(a_res) + kt * GR_TILE_BYTES;
                if (!args.tma2d) {
                    tma_load_3d(dst, mapA, resa_bar(), 0, kt * GR_BK, tm * 2);
                } else {
                    tma_load_2d(dst, mapA, resa_bar(), (tm * 2) * 16, kt * GR_BK);
                    tma_load_2d(dst + GR_SLAB_BYTES, mapA, resa_bar(), (tm * 2 + 1) * 16, kt * GR_BK);
                }
            }
        }
        if (tn >= args.tiles_n) return;
        int stage = 0;
        uint32_t phase = 0;
        for (int s = 0; s < nsteps; ++s) {
            const int ti = args.first_task + s;
            const Task* tk = args.tasks + ti;
            if (tk->ktiles > 0) {
                wait_counter(args.panel_done + (size_t)(ti - 1) * args.panel_stride + tn, args.tiles_m, args.error_flag);
                fence_proxy_async();
                const CUtensorMap* mapB = args.maps + tk->mapB;
                for (int kt = 0; kt < ktiles; ++kt) {
                    mbar_wait(empty_bar(g, stage), phase ^ 1);
                    const uint32_t dst = smem_u32(ring0) + (g * GR_STAGES + stage) * GR_TILE_BYTES;
                    mbar_arrive_expect_tx(full_bar(g, stage), GR_TILE_BYTES);
                    if (!args.tma2d) {
                        tma_load_3d(dst, mapB, full_bar(g, stage), 0, kt * GR_BK, tn * 2);
                    } else {
                        tma_load_2d(dst, mapB, full_bar(g, stage), (tn * 2) * 16, kt * GR_BK);
                        tma_load_2d(dst + GR_SLAB_BYTES, mapB, full_bar(g, stage), (tn * 2 + 1) * 16, kt * GR_BK);
                    }
                    if (++stage == GR_STAGES) { stage = 0; phase ^= 1; }
                }
            }
            // the consumer warps arrive after their stores (release, CTA scope); one gpu-scope fence makes the
            // tile visible device-wide, then the panel counter is bumped
            mbar_wait(stored_bar(g), (uint32_t)(s & 1));
            fence_acq_rel_gpu();
            red_relaxed_gpu_add(args.panel_done + (size_t)ti * args.panel_stride + tn, 1);
        }
        return;
    }

    // ==================================== consumer group g ====================================
    const int g = warp / GR_GROUP_WARPS;
    const int wg = warp % GR_GROUP_WARPS;
    const int wm = wg >> 1, wn = wg & 1;
    const int tn = 2 * pair + g;
    if (tn >= args.tiles_n) return;
    const int gq = lane >> 2, t = lane & 3;
    // fragment offsets inside an 8 KB operand block, same layout as gemm_dmma.cuh (k4-step j: jh = j>>1,
    // par = j&1, k-row 8 jh + par + 2t; column c in slab c>>4, 16-byte chunk ((c&15)>>1) ^ (row&7))
    uint32_t off[2];
#pragma unroll
    for (int par = 0; par < 2; ++par) {
        const uint32_t x = par + 2 * t;
        off[par] = x * 128 + ((((uint32_t)gq >> 1) ^ x) << 4) + (gq & 1) * 8;
    }
    const uint32_t aoff_w = wm * GR_SLAB_BYTES, boff_w = wn * GR_SLAB_BYTES;
    const int row0 = tm * GR_BM + wm * 16 + gq;
    const int col0 = tn * GR_BN + wn * 16 + 2 * t;
    const bool tracing = (args.trace != nullptr) && lane == 0 && wg == 0;

    mbar_wait(resa_bar(), 0);
    int stage = 0;
    uint32_t phase = 0;

    for (int s = 0; s < nsteps; ++s) {
        const int ti = args.first_task + s;
        const Task* tk = args.tasks + ti;
        unsigned long long t_desc = 0, t_first = 0, t_kend = 0;
        if (tracing) t_desc = global_ns();
        double acc[2][2][2];
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

        // ---- prologue: low-order sum (Eq. 21) into registers of its own (added in the epilogue; starting the
        // accumulator from it costs accuracy, see gemm_dmma.cuh); the baby block is complete (stream order), so this
        // overlaps the wait for the previous step of this panel ----
        double pre[2][2][2];
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j) pre[i][j][0] = pre[i][j][1] = 0.0;
        const int ns = tk->sum_count;
        if (ns > 0) {
            const double* coef = tk->coef;
            const long long lds = tk->lds, sstride = tk->sum_stride;
            const double* sb = tk->sum_base + (long long)row0 * lds + col0;
            int q = 0;
            for (; q + 7 < ns; q += 8) {  // eight operands in flight
                double w[8];
                double2 v[8][2][2];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    w[u] = __ldg(coef + q + u);
                    const double* pu = sb + (long long)(q + u) * sstride;
#pragma unroll
                    for (int i = 0; i < 2; ++i)
#pragma unroll
                        for (int j = 0; j < 2; ++j) {
                            const bool in = (row0 + i * 8 < N) && (col0 + j * 8 < N);
                            v[u][i][j] = in ? __ldcg(reinterpret_cast<const double2*>(pu + (long long)(i * 8) * lds + j * 8)) : make_double2(0.0, 0.0);
                        }
                }
#pragma unroll
                for (int u = 0; u < 8; ++u)
#pragma unroll
                    for (int i = 0; i < 2; ++i)
#pragma unroll
                        for (int j = 0; j < 2; ++j) {
                            pre[i][j][0] = fma(w[u], v[u][i][j].x, pre[i][j][0]);
                            pre[i][j][1] = fma(w[u], v[u][i][j].y, pre[i][j][1]);
                        }
            }
            for (; q < ns; ++q) {
                const double w0 = __ldg(coef + q);
                const double* pu = sb + (long long)q * sstride;
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 2; ++j)
                        if ((row0 + i * 8 < N) && (col0 + j * 8 < N)) {
                            const double2 v = __ldcg(reinterpret_cast<const double2*>(pu + (long long)(i * 8) * lds + j * 8));
                            pre[i][j][0] = fma(w0, v.x, pre[i][j][0]);
                            pre[i][j][1] = fma(w0, v.y, pre[i][j][1]);
                        }
            }
        }
        {
            double diag = tk->diag_const;
            if (tk->diag_ptr != nullptr) diag += __ldg(tk->diag_ptr);
            if (diag != 0.0) {
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        const int r = row0 + i * 8, c = col0 + j * 8;
                        if (r == c) pre[i][j][0] += diag;
                        if (r == c + 1) pre[i][j][1] += diag;
                    }
            }
        }

        // ---- K loop: A from the resident block, B from this group's ring; C fetched at the first full barrier ----
        const double* Cp = tk->C;
        const long long ldc = tk->ldc;
        double creg[2][2][2];
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j) creg[i][j][0] = creg[i][j][1] = 0.0;
        const int kts = tk->ktiles;
        // Stagger: in lockstep both groups would share the DMMA pipe during their K loops and then both sit in
        // the latency part of the chain.  Group 1 therefore starts its first K loop when group 0 is half way
        // through its own; the offset persists (the two panel families are independent chains), so from then on
        // one group's K loop covers the other's store -> flag -> poll -> TMA latency.
        if (s == 1 && g == 1 && kts > 0) mbar_wait(stagger_bar(), 0);
        int prev_stage = -1;  // stages are released one iteration late (see gemm_dmma.cuh: the arrive must not
                              // overtake ld.shared that are still in flight)
        for (int kt = 0; kt < kts; ++kt) {
            if (s == 1 && g == 0 && kt == kts / 2) {
                __syncwarp();
                if (lane == 0) mbar_arrive(stagger_bar());
            }
            mbar_wait(full_bar(g, stage), phase);
            if (prev_stage >= 0) {
                __syncwarp();
                if (lane == 0) mbar_arrive(empty_bar(g, prev_stage));
            }
            if (kt == 0) {
                if (tracing) t_first = global_ns();
                if (Cp != nullptr) {  // workspace matrix: even ld, 16-byte aligned rows, zero pad columns
#pragma unroll
                    for (int i = 0; i < 2; ++i)
#pragma unroll
                        for (int j = 0; j < 2; ++j)
                            if ((row0 + i * 8 < N) && (col0 + j * 8 < N)) {
                                const double2 v = __ldcg(reinterpret_cast<const double2*>(Cp + (long long)(row0 + i * 8) * ldc + col0 + j * 8));
                                creg[i][j][0] = v.x;
                                creg[i][j][1] = v.y;
                            }
                }
            }
            const uint8_t* sa = a_res + kt * GR_TILE_BYTES + aoff_w;
            const uint8_t* sbm = ring0 + (g * GR_STAGES + stage) * GR_TILE_BYTES + boff_w;
#pragma unroll
            for (int j = 0; j < GR_BK / 4; ++j) {
                const int jh = j >> 1, par = j & 1;
                double a[2], b[2];
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    a[i] = *reinterpret_cast<const double*>(sa + ((off[par] ^ ((i & 1) << 6)) + jh * 1024));
                    b[i] = *reinterpret_cast<const double*>(sbm + ((off[par] ^ ((i & 1) << 6)) + jh * 1024));
                }
#pragma unroll
                for (int im = 0; im < 2; ++im)
#pragma unroll
                    for (int jn = 0; jn < 2; ++jn) dmma_884(acc[im][jn][0], acc[im][jn][1], a[im], b[jn]);
            }
            prev_stage = stage;
            if (++stage == GR_STAGES) { stage = 0; phase ^= 1; }
        }
        if (prev_stage >= 0) {
            int dep = 0;
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) dep ^= __double2hiint(acc[i][j][0]) ^ __double2hiint(acc[i][j][1]);
            __syncwarp();
            if (lane == 0) mbar_arrive_dep(empty_bar(g, prev_stage), dep);
        }
        if (tracing) t_kend = global_ns();

        // ---- epilogue: Out = alpha acc + beta C ----
        const double alpha = tk->alpha, beta = (Cp != nullptr) ? tk->beta : 0.0;
        double* Out = tk->out_is_user ? args.userD : tk->Out;
        const long long ldo = tk->out_is_user ? args.ldD : tk->ldo;
        const bool vec = ((ldo & 1) == 0) && ((reinterpret_cast<uintptr_t>(Out) & 15) == 0);
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const int r = row0 + i * 8;
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const int c = col0 + j * 8;
                const double o0 = fma(beta, creg[i][j][0], alpha * acc[i][j][0]) + pre[i][j][0];
                const double o1 = fma(beta, creg[i][j][1], alpha * acc[i][j][1]) + pre[i][j][1];
                if (r < N && c < N) {
                    double* p = Out + (long long)r * ldo + c;
                    if (vec && c + 1 < N) {
                        __stcg(reinterpret_cast<double2*>(p), make_double2(o0, o1));
                    } else {
                        __stcg(p, o0);
                        if (c + 1 < N) __stcg(p + 1, o1);
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(stored_bar(g));  // hand the publication over to the producer warp
        if (tracing) {
            TraceRec r;
            r.task = ti; r.tm = tm; r.tn = tn; r.sm = sm_id();
            r.t_claim = t_desc; r.t_desc = t_desc; r.t_first = t_first; r.t_kend = t_kend; r.t_done = global_ns();
            args.trace[args.trace_base + ((size_t)s * args.tiles_n + tn) * args.tiles_m + tm] = r;
        }
    }
}

}  // namespace chebdm
