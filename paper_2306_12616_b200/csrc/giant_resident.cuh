// giant_resident.cuh -- giant steps (Eq. 4, or its Clenshaw form, reading A6) for
// small N (N <= 512), as ONE persistent launch in which
//   * every CTA keeps its 32-row block of the multiplier Y = T_k resident in shared memory for all p-1
//     products (the A operand never changes along the chain: 32 x Kpad x 8 B <= 128 KB), so a step only
//     streams the B operand (the previous accumulator panel) from L2;
//   * every CTA owns TWO column panels (32 columns each).  Column panels are independent chains (step l of panel
//     tn needs only panel tn of step l+1), and the 8 consumer warps alternate between them: while the result of
//     panel a travels through the latency part of its chain (store -> fence -> flag -> poll of the other 15 CTAs
//     of that panel -> TMA round trip, ~3.5 us) the DMMA pipe works on panel b, whose operand stages its own
//     producer warp has prefetched into its own ring;
//   * the low-order sums G_l / S_j of Eq. (21) are formed once at kernel start by the CTA that
//     consumes them (each T_i tile read once for all p sums, results parked in L2) while the multiplier block is
//     being loaded, and each step's G tile is prefetched into registers one tile ahead;
//   * completion is published by the panel's producer warp (mbarrier hand-off, one gpu fence, one relaxed
//     increment), so the consumer warps go straight on to the other panel.
// This replaces, for the serial part of the solve, the stream-level concurrency of PAPER.md:228-232 (which the
// paper found to help only below N ~ 1000).  Measured per giant step at N = 500: DESIGN.md section 6.
//
// Work assignment is static: CTA b handles row block tm = b % tiles_m and the panels tn = 2 (b / tiles_m) + g,
// g = 0, 1.  All CTAs must be co-resident (cooperative launch); they synchronise only through the per-panel
// completion counters of gemm_dmma.cuh.
//
// Symmetric mode (args.sym, the default): every B_l is a polynomial of X, hence symmetric, so the grid
// is the T (T + 1) / 2 lower-triangle tiles (136 at N = 500), ONE tile per CTA.  The CTA still keeps its 32 rows of
// T_k resident and streams its panel; it mirrors its tile into (tn, tm) with an in-warp shuffle transpose, and because
// a panel now also receives mirrored blocks from other panels a step waits for the whole previous step (one counter
// per step).  Half the flops per step and half the sums per CTA: 12.2 -> 8.7 us per giant step at N = 500.
#pragma once
#include "gemm_dmma.cuh"

namespace chebdm {

constexpr int GR_BM = 32, GR_BN = 32, GR_BK = 32, GR_STAGES = 5;
constexpr int GR_SLAB_BYTES = GR_BK * 128;               // 4 KB: 16 columns x 32 k-rows
constexpr int GR_TILE_BYTES = 2 * GR_SLAB_BYTES;         // 8 KB: one 32-column operand block of one k-tile
constexpr int GR_CONSUMER_WARPS = 8;                     // 2 k-halves x (2 x 2 warps of 16 x 16) on a 32 x 32 tile
constexpr int GR_THREADS = (GR_CONSUMER_WARPS + 2) * 32;   // consumer warps + one producer warp per panel
constexpr int GR_SUM_CHUNK = 16;                         // low-order sums formed per pass over the baby block
constexpr int GR_MAX_KTILES = 16;                        // N <= 512

struct GiantArgs {
    const Task* tasks;       // giant tasks: tasks[(first_task + s) * task_stride], s = 0..nsteps-1 (s = 0 is the product-free step)
    const CUtensorMap* maps;
    int first_task, nsteps, task_stride;
    int N, ktiles;
    int tiles_m, tiles_n;    // 32-row blocks, 32-column panels
    int* panel_done;         // [step][panel] completion counters (target tiles_m)
    int panel_stride;
    double* userD;
    long long ldD;
    int tma2d;
    int* error_flag;
    TraceRec* trace;         // nullable; record index = trace_base + (s * tiles_n + tn) * tiles_m + tm
    int trace_base;
    // low-order sums, formed in the kernel: G_l = coefT[l*k] I + sum_{i=1}^{k-1} coefT[l*k + i] T_i  (l = nsteps-1-s)
    const double* coefT;     // g (Clenshaw) or d (Eq. 4) table, layout [l][i]
    const double* Tbase;     // T_1; T_i at Tbase + (i-1) * mat_stride
    double* Gbase;           // G_0; G_l at Gbase + l * mat_stride
    long long mat_stride, ld;
    int k;
    int sym;                 // 1: symmetric-tile skipping: grid = lower-triangle tiles (tm >= tn), one tile per CTA, the
                             // tile is mirrored into (tn, tm), a step waits for the whole previous step
};

inline int giant_resident_smem_bytes(int ktiles) {
    return ktiles * GR_TILE_BYTES + 2 * GR_STAGES * GR_TILE_BYTES + 256 + 2 * 128 * 8 * 8 + 1024;  // + k-split scratch
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

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        mbar_init(resa_bar(), 1);
        for (int g = 0; g < 2; ++g) {
            for (int s = 0; s < GR_STAGES; ++s) {
                mbar_init(full_bar(g, s), 1);
                mbar_init(empty_bar(g, s), GR_CONSUMER_WARPS / 2);  // the k-half that reads the stage
            }
            mbar_init(stored_bar(g), GR_CONSUMER_WARPS / 2);  // the four epilogue warps
        }
        fence_mbar_init();
    }
    __syncthreads();

    // tile assignment: full mode -> row block tm, panels 2 pair + {0, 1}; symmetric mode -> one lower-triangle tile
    int tm, pair, tn_sym = 0;
    if (!args.sym) {
        tm = blockIdx.x % args.tiles_m;
        pair = blockIdx.x / args.tiles_m;
    } else {
        int b = blockIdx.x;
        while (b >= args.tiles_m - tn_sym) { b -= args.tiles_m - tn_sym; ++tn_sym; }  // panel-major: panel tn holds tm = tn..T-1
        tm = tn_sym + b;
        pair = 0;
    }
    const int tn_of[2] = {args.sym ? tn_sym : 2 * pair, args.sym ? args.tiles_n : 2 * pair + 1};  // panel of group g (>= tiles_n: none)
    const int dep_target = args.sym ? (args.tiles_m * (args.tiles_m + 1)) / 2 : args.tiles_m;
    const int N = args.N;
    const int nsteps = args.nsteps;

    if (warp >= GR_CONSUMER_WARPS) {
        // =============================== producer warp of panel g ===============================
        const int g = warp - GR_CONSUMER_WARPS;
        const int tn = tn_of[g];
        const int ctr = args.sym ? 0 : tn;  // symmetric mode: one counter per step (every tile feeds every panel)
        if (lane != 0) return;
        if (g == 0) {
            // resident A: rows [tm*32, tm*32+32) of Y = T_k as [k][column] blocks (Y is symmetric)
            const Task* t1 = args.tasks + (size_t)(args.first_task + (nsteps > 1 ? 1 : 0)) * args.task_stride;
            const CUtensorMap* mapA = args.maps + t1->mapA;
            fence_tensormap_acquire(mapA);
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
            const Task* tk = args.tasks + (size_t)(args.first_task + s) * args.task_stride;
            if (tk->ktiles > 0) {
                wait_counter(args.panel_done + (size_t)(s - 1) * args.panel_stride + ctr, dep_target, args.error_flag);
                fence_proxy_async_global();
                const CUtensorMap* mapB = args.maps + tk->mapB;
                if (s <= 3) fence_tensormap_acquire(mapB);  // the three rotating buffers take turns as operand B
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
            red_relaxed_gpu_add(args.panel_done + (size_t)s * args.panel_stride + ctr, 1);
        }
        return;
    }


    // ======================================= consumer warps =======================================
    // Products: the 8 warps form 2 k-halves x (2 x 2 warps of 16 x 16); warp w takes the k4-steps [4 kh, 4 kh + 4) of
    // every stage (kh = w >> 2) and the two halves are added through shared memory at the end of the K loop.  (16 x 8
    // warp tiles without the k-split need 1.5 ld.shared per DMMA and only two accumulator chains per warp: measured
    // 25 % slower.)  The sums pass below uses all 8 warps on 16 x 8 sub-tiles.
    const int kh = warp >> 2, wq = warp & 3;
    const int wm = wq >> 1, wn = wq & 1;
    const int gq = lane >> 2, t = lane & 3;
    // fragment offsets inside an 8 KB operand block, same layout as gemm_dmma.cuh (k4-step j: jh = j>>1,
    // par = j&1, k-row 8 jh + par + 2t; column c in slab c>>4, 16-byte chunk ((c&15)>>1) ^ (row&7))
    uint32_t aoff[2], boff[2];
#pragma unroll
    for (int par = 0; par < 2; ++par) {
        const uint32_t x = par + 2 * t;
        const uint32_t lo = x * 128 + ((((uint32_t)gq >> 1) ^ x) << 4) + (gq & 1) * 8;
        aoff[par] = wm * GR_SLAB_BYTES + lo;
        boff[par] = wn * GR_SLAB_BYTES + lo;
    }
    const int row0 = tm * GR_BM + wm * 16 + gq;
    const int npanels = (tn_of[1] < args.tiles_n) ? 2 : 1;
    int colp[2];
    colp[0] = tn_of[0] * GR_BN + wn * 16 + 2 * t;
    colp[1] = tn_of[1] * GR_BN + wn * 16 + 2 * t;
    const bool tracing = (args.trace != nullptr) && threadIdx.x == 0;
    const long long ld = args.ld;
    double* scratch = reinterpret_cast<double*>(ring0 + 2 * GR_STAGES * GR_TILE_BYTES + 256);  // [2][128 threads][8]

    // ---- low-order sums of this CTA's tiles, all steps (Eq. 21): every T_i element is read once per chunk of
    // GR_SUM_CHUNK sums; each thread writes (and later re-reads) only its own elements, so no synchronisation is
    // needed beyond program order.  Runs while the producer warp loads the resident multiplier block. ----
    {
        double* s_coef = reinterpret_cast<double*>(ring0);  // [k][GR_SUM_CHUNK]; the rings are idle until step 1
        const int k = args.k;
        const int srow0 = tm * GR_BM + (warp >> 2) * 16 + gq;  // 16 x 8 sub-tile of warp (warp >> 2, warp & 3)
        const int scol[2] = {tn_of[0] * GR_BN + (warp & 3) * 8 + 2 * t, tn_of[1] * GR_BN + (warp & 3) * 8 + 2 * t};
        for (int l0 = 0; l0 < nsteps; l0 += GR_SUM_CHUNK) {
            const int nl = min(GR_SUM_CHUNK, nsteps - l0);
            named_bar_sync(1, GR_CONSUMER_WARPS * 32);
            for (int e = threadIdx.x; e < k * GR_SUM_CHUNK; e += GR_CONSUMER_WARPS * 32) {
                const int i = e / GR_SUM_CHUNK, q = e - i * GR_SUM_CHUNK;
                s_coef[e] = (q < nl) ? __ldg(args.coefT + (size_t)(l0 + q) * k + i) : 0.0;
            }
            named_bar_sync(1, GR_CONSUMER_WARPS * 32);
            for (int g = 0; g < npanels; ++g) {
                const int c = scol[g];
                double2 sum[GR_SUM_CHUNK][2];
#pragma unroll
                for (int q = 0; q < GR_SUM_CHUNK; ++q) sum[q][0] = sum[q][1] = make_double2(0.0, 0.0);
                const bool in0 = (srow0 < N) && (c < N), in1 = (srow0 + 8 < N) && (c < N);
                const double* src = args.Tbase + (long long)srow0 * ld + c;
                int i = 1;
                for (; i + 4 < k; i += 5) {  // five operands (10 loads) in flight
                    double2 v[5][2];
#pragma unroll
                    for (int u = 0; u < 5; ++u) {
                        const double* pu = src + (long long)(i - 1 + u) * args.mat_stride;
                        v[u][0] = in0 ? __ldcg(reinterpret_cast<const double2*>(pu)) : make_double2(0.0, 0.0);
                        v[u][1] = in1 ? __ldcg(reinterpret_cast<const double2*>(pu + 8 * ld)) : make_double2(0.0, 0.0);
                    }
#pragma unroll
                    for (int u = 0; u < 5; ++u)
#pragma unroll
                        for (int q = 0; q < GR_SUM_CHUNK; ++q) {
                            const double w = s_coef[(i + u) * GR_SUM_CHUNK + q];
                            sum[q][0].x = fma(w, v[u][0].x, sum[q][0].x);
                            sum[q][0].y = fma(w, v[u][0].y, sum[q][0].y);
                            sum[q][1].x = fma(w, v[u][1].x, sum[q][1].x);
                            sum[q][1].y = fma(w, v[u][1].y, sum[q][1].y);
                        }
                }
                for (; i < k; ++i) {
                    const double* pu = src + (long long)(i - 1) * args.mat_stride;
                    const double2 v0 = in0 ? __ldcg(reinterpret_cast<const double2*>(pu)) : make_double2(0.0, 0.0);
                    const double2 v1 = in1 ? __ldcg(reinterpret_cast<const double2*>(pu + 8 * ld)) : make_double2(0.0, 0.0);
#pragma unroll
                    for (int q = 0; q < GR_SUM_CHUNK; ++q) {
                        const double w = s_coef[i * GR_SUM_CHUNK + q];
                        sum[q][0].x = fma(w, v0.x, sum[q][0].x);
                        sum[q][0].y = fma(w, v0.y, sum[q][0].y);
                        sum[q][1].x = fma(w, v1.x, sum[q][1].x);
                        sum[q][1].y = fma(w, v1.y, sum[q][1].y);
                    }
                }
#pragma unroll
                for (int q = 0; q < GR_SUM_CHUNK; ++q) {
                    if (q < nl) {
                        const double d0 = s_coef[q];  // coefficient of T_0 = I
                        double* dst = args.Gbase + (long long)(l0 + q) * args.mat_stride + (long long)srow0 * ld + c;
                        if (in0) {
                            double2 o = sum[q][0];
                            if (srow0 == c) o.x += d0;
                            if (srow0 == c + 1) o.y += d0;
                            __stcg(reinterpret_cast<double2*>(dst), o);
                        }
                        if (in1) {
                            double2 o = sum[q][1];
                            if (srow0 + 8 == c) o.x += d0;
                            if (srow0 + 8 == c + 1) o.y += d0;
                            __stcg(reinterpret_cast<double2*>(dst + 8 * ld), o);
                        }
                    }
                }
            }
        }
        // The sums are re-read by other threads of this CTA (different thread mapping): CTA barrier.  s_coef lives in
        // ring memory: the first TMA into a ring is issued only after this CTA's own step-0 tile has been published
        // (the producer waits for the panel counter and runs fence.proxy.async), i.e. after this point.
        named_bar_sync(1, GR_CONSUMER_WARPS * 32);
    }

    mbar_wait(resa_bar(), 0);
    int stage[2] = {0, 0};
    uint32_t phase[2] = {0u, 0u};
    int tile_no = 0;

    // G tile of (step s, panel g): this thread's 2 x 2 fragments (epilogue warps only); plan-owned matrices (even ld)
    auto load_pre = [&](int s, int g, double2 (&pv)[2][2]) {
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j) pv[i][j] = make_double2(0.0, 0.0);
        if (kh != 0 || s >= nsteps || g >= npanels) return;
        const Task* tk = args.tasks + (size_t)(args.first_task + s) * args.task_stride;
        if (tk->sum_count <= 0) return;
        const double* sb = tk->sum_base + (long long)row0 * tk->lds + colp[g];
#pragma unroll
        for (int i = 0; i < 2; ++i)
#pragma unroll
            for (int j = 0; j < 2; ++j)
                if (row0 + i * 8 < N && colp[g] + j * 8 < N)
                    pv[i][j] = __ldcg(reinterpret_cast<const double2*>(sb + (long long)(i * 8) * tk->lds + j * 8));
    };
    double2 pre[2][2];
    load_pre(0, 0, pre);

    for (int s = 0; s < nsteps; ++s) {
        const int ti = args.first_task + s;
        const Task* tk = args.tasks + (size_t)ti * args.task_stride;
        const int kts = tk->ktiles;
        const double alpha = tk->alpha;
        const double* Cp = tk->C;
        const double beta = (Cp != nullptr) ? tk->beta : 0.0;
        const long long ldc = tk->ldc;
        double* Out = tk->out_is_user ? args.userD : tk->Out;
        const long long ldo = tk->out_is_user ? args.ldD : tk->ldo;
        const bool vec = ((ldo & 1) == 0) && ((reinterpret_cast<uintptr_t>(Out) & 15) == 0);
#pragma unroll
        for (int g = 0; g < 2; ++g) {
            if (g >= npanels) break;
            const int tn = tn_of[g];
            const int col0 = colp[g];
            unsigned long long t_desc = 0, t_first = 0, t_kend = 0;
            if (tracing) t_desc = global_ns();
            double acc[2][2][2];
            double2 creg[2][2], nxt[2][2];
#pragma unroll
            for (int i = 0; i < 2; ++i)
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    acc[i][j][0] = acc[i][j][1] = 0.0;
                    creg[i][j] = nxt[i][j] = make_double2(0.0, 0.0);
                }
            const int ns_ = (g + 1 < npanels) ? s : s + 1, ng_ = (g + 1 < npanels) ? g + 1 : 0;  // next tile
            if (kts == 0) load_pre(ns_, ng_, nxt);
            int prev_stage = -1;  // stages are released one iteration late (see gemm_dmma.cuh)
            // the two k-halves take ALTERNATE k-tiles (kh = kt & 1), all eight k4-steps of their stages: the two warps of a
            // scheduler sub-partition (w, w + 4) then never wait behind the same stage barrier together
            for (int kt = 0; kt < kts; ++kt) {
                if ((kt & 1) == kh) {
                    mbar_wait(full_bar(g, stage[g]), phase[g]);
                    if (kt == 0) {
                        // the late dependencies of this tile hold: fetch C now, and the next tile's G one tile ahead
                        if (tracing) t_first = global_ns();
                        if (Cp != nullptr) {  // workspace matrix: even ld, 16-byte aligned rows, zero pad columns (kh == 0 here)
#pragma unroll
                            for (int i = 0; i < 2; ++i)
#pragma unroll
                                for (int j = 0; j < 2; ++j)
                                    if (row0 + i * 8 < N && col0 + j * 8 < N)
                                        creg[i][j] = __ldcg(reinterpret_cast<const double2*>(Cp + (long long)(row0 + i * 8) * ldc + col0 + j * 8));
                        }
                        load_pre(ns_, ng_, nxt);
                    }
                    const uint8_t* sa = a_res + kt * GR_TILE_BYTES;
                    const uint8_t* sbm = ring0 + (g * GR_STAGES + stage[g]) * GR_TILE_BYTES;
#pragma unroll
                    for (int j = 0; j < GR_BK / 4; ++j) {
                        const int jh = j >> 1, par = j & 1;
                        double a[2], b[2];
#pragma unroll
                        for (int i = 0; i < 2; ++i) {
                            a[i] = *reinterpret_cast<const double*>(sa + ((aoff[par] ^ ((i & 1) << 6)) + jh * 1024));
                            b[i] = *reinterpret_cast<const double*>(sbm + ((boff[par] ^ ((i & 1) << 6)) + jh * 1024));
                        }
                        if (j == 0 && prev_stage >= 0) {  // previous stage back to the producer (after this stage's barrier)
                            __syncwarp();
                            if (lane == 0) mbar_arrive(empty_bar(g, prev_stage));
                        }
#pragma unroll
                        for (int im = 0; im < 2; ++im)
#pragma unroll
                            for (int jn = 0; jn < 2; ++jn) dmma_884(acc[im][jn][0], acc[im][jn][1], a[im], b[jn]);
                    }
                    prev_stage = stage[g];
                }
                if (++stage[g] == GR_STAGES) { stage[g] = 0; phase[g] ^= 1; }
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

            // ---- add the two k-halves (double-buffered scratch; the barrier of the next tile separates reuse) ----
            double* sc = scratch + (tile_no & 1) * (128 * 8) + (wq * 32 + lane) * 8;
            if (kh == 1) {
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 2; ++j)
                        *reinterpret_cast<double2*>(sc + (i * 2 + j) * 2) = make_double2(acc[i][j][0], acc[i][j][1]);
            }
            named_bar_sync(1, GR_CONSUMER_WARPS * 32);
            ++tile_no;
            if (kh == 0) {
                // ---- epilogue: Out = alpha (acc_lo + acc_hi) + beta C + G ----
#pragma unroll
                for (int i = 0; i < 2; ++i) {
                    const int r = row0 + i * 8;
#pragma unroll
                    for (int j = 0; j < 2; ++j) {
                        const int c = col0 + j * 8;
                        const double2 hi = *reinterpret_cast<const double2*>(sc + (i * 2 + j) * 2);
                        const double o0 = fma(beta, creg[i][j].x, alpha * (acc[i][j][0] + hi.x)) + pre[i][j].x;
                        const double o1 = fma(beta, creg[i][j].y, alpha * (acc[i][j][1] + hi.y)) + pre[i][j].y;
                        acc[i][j][0] = o0;
                        acc[i][j][1] = o1;
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
                if (args.sym && tm > tn) {
                    // mirror the tile into (tn, tm): every 8x8 block is transposed inside the warp (lane (g, t) of the
                    // transposed block takes C[2t][g], C[2t+1][g] from lanes (2t, g>>1), (2t+1, g>>1)) and stored
                    // row-contiguously, like the direct store
                    const int src0 = (2 * t) * 4 + (gq >> 1), src1 = src0 + 4;
#pragma unroll
                    for (int i = 0; i < 2; ++i)
#pragma unroll
                        for (int j = 0; j < 2; ++j) {
                            const double a0 = __shfl_sync(0xffffffffu, acc[i][j][0], src0), a1 = __shfl_sync(0xffffffffu, acc[i][j][1], src0);
                            const double b0 = __shfl_sync(0xffffffffu, acc[i][j][0], src1), b1 = __shfl_sync(0xffffffffu, acc[i][j][1], src1);
                            const double w0 = (gq & 1) ? a1 : a0, w1 = (gq & 1) ? b1 : b0;
                            const int rr = tn * GR_BN + wn * 16 + j * 8 + gq, cc = tm * GR_BM + wm * 16 + i * 8 + 2 * t;
                            if (rr < N && cc < N) {
                                double* p = Out + (long long)rr * ldo + cc;
                                if (vec && cc + 1 < N) {
                                    __stcg(reinterpret_cast<double2*>(p), make_double2(w0, w1));
                                } else {
                                    __stcg(p, w0);
                                    if (cc + 1 < N) __stcg(p + 1, w1);
                                }
                            }
                        }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(stored_bar(g));  // hand the publication over to the panel's producer warp
                if (tracing) {
                    TraceRec r;
                    r.task = ti; r.tm = tm; r.tn = tn; r.sm = sm_id();
                    r.t_claim = t_desc; r.t_desc = t_desc; r.t_first = t_first; r.t_kend = t_kend; r.t_done = global_ns();
                    args.trace[args.trace_base + ((size_t)s * args.tiles_n + tn) * args.tiles_m + tm] = r;
                }
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int j = 0; j < 2; ++j) pre[i][j] = nxt[i][j];
            }
        }
    }
}

}  // namespace chebdm
