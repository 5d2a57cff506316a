// gemm_dmma.cuh -- persistent grouped FP64 GEMM for sm_100a (north_star items 2 and 3).
//
// One launch runs a list of "tasks".  A task is one product of the recurrence with its fused epilogue
//
//     Out = alpha * (A^T B) + beta * C + sum_{i<ns} coef[i] * S_i + diag * I
//
// which covers  T_{a+b} = 2 T_a T_b - T_|a-b|          (Eq. 7, 22-23, Alg. 1),
//               acc    <- S_j + T_k acc                 (Eq. 4; S_j of Eq. 21, :196-201)
//           and B_l     = G_l + 2 T_k B_{l+1} - B_{l+2} (Clenshaw form of Eq. 4, reading A6),
// the low-order sums S_j / G_l = sum_i coef_i T_i being formed in registers by the epilogue, so the
// "matrix additions" of PAPER.md:234 never make a separate pass over HBM.  All operands of the method
// are symmetric polynomials of X, so A^T = A: both operands are fetched as [k][column] tiles.
//
// Hardware mapping.  sm_100a has no tcgen05 kind::f64; FP64 tensor work is mma.sync.m8n8k4 -> SASS
// DMMA.8x8x4 (measured 37.17 TFLOP/s = 64 FMA/clk/SM, one DMMA per 16 clk per SM sub-partition).
// Operand tiles are staged by TMA (cp.async.bulk.tensor.3d, 128-byte swizzle) into a ring of shared-
// memory stages guarded by full/empty mbarriers; one producer warp issues TMA, the consumer warps each
// own a 32x32 accumulator tile in registers.  The swizzled layout plus an interleaved k-assignment
// (lane t of a DMMA takes k-rows {par+2t}) makes every 64-bit ld.shared bank-conflict free.
//
// Scheduling.  CTAs are persistent: the producer lane claims work items (task, tile) from a global
// counter in topological order, waits on global completion counters (whole task, one column panel of a
// task, or a whole group of tasks), then streams the tile's K loop.  Claiming in order makes the spin
// waits deadlock-free whatever the residency.  This replaces the paper's stream-level concurrency
// (Alg. 1 "sync streams()").
#pragma once
#include "common.cuh"

namespace chebdm {

constexpr int TILE_RING = 2;            // producer run-ahead (tile descriptors in flight)
constexpr int MAX_DEPS = 4;
constexpr long long WATCHDOG_CLOCKS = 8000000000ll;

// DEP_TASK: every tile of a task; DEP_PANEL_N: the tiles of one column panel of a task (non-symmetric tasks: a panel is
// written by its own tiles only); DEP_PANEL_SYM: everything a SYMMETRIC task writes into one column panel -- its own tiles
// plus the tiles of the row block(s) whose mirror lands there (target: LaunchArgs::sym_panel_target[panel]).
enum DepKind : int { DEP_NONE = 0, DEP_TASK = 1, DEP_PANEL_N = 2, DEP_PANEL_SYM = 3 };

struct Task {
    // operands (indices into the tensor-map table); ktiles == 0 => no product, epilogue only
    int mapA, mapB;
    int ktiles;
    int tiles_m, tiles_n;
    int sym;                 // 1: the result is symmetric (every operand is a polynomial of X): only the tiles that touch
                             // the lower triangle are work items, each mirrors its blocks into the skipped tiles
    int nitems;              // work items of this task (tiles_m * tiles_n, or the lower-triangle count when sym)
    int slot;                // matrix of the batch this task belongs to (0 for single solves)
    int out_is_user;         // Out = the user's D of this slot (pointer/ld come from the launch parameters)
    int kchunks;             // >= 1: the K loop runs over kchunks operand pairs (mapA + c, mapB + c), ktiles k-tiles
                             // each: one long-K product  sum_c A_c^T B_c  (flat giant step)
    int ndeps;
    int ndeps_early;         // deps [0, ndeps_early) guard the operands of the low-order sum (read by the consumer
                             // warps BEFORE the K loop); the rest guard the TMA operands and C
    int dep_kind[MAX_DEPS];
    int dep_idx[MAX_DEPS];   // task index inside the table of this launch (DEP_TASK, DEP_PANEL_N)
    int dep_target[MAX_DEPS];  // counter value that means "complete" (tiles of the task / panel)
    double alpha, beta;
    const double* C;         // nullable
    long long ldc;
    double* Out;
    long long ldo;
    const double* sum_base;  // S_i = sum_base + i * sum_stride   (same ld as the workspace)
    long long sum_stride;
    long long lds;
    int sum_count;
    const double* coef;      // coef[i], i < sum_count (device memory, written by the coefficient kernel)
    const double* diag_ptr;  // nullable: coefficient of T_0 = I
    double diag_const;
};

struct TraceRec;

// A launch runs the tasks of one table.  The table holds, for every "level task" lt (one product of the method, in
// topological order), one task per matrix of the batch: index lt * maxb + slot.  A launch covers the level tasks
// [lt_begin, lt_end) of the slots [0, nb); every task of a table has the same number of work items, so work item w of
// the launch is tile (w % items_per_task) of task ((w / items_per_task) / nb, (w / items_per_task) % nb): items are
// claimed level by level and, inside a level, matrix by matrix -- the independent products of different matrices
// fill the machine where one small matrix cannot.
struct LaunchArgs {
    const Task* tasks;       // table
    const CUtensorMap* maps;
    int* work_counter;       // claimed-items counter of this launch
    int* task_done;          // [table tasks]
    int* panel_done;         // [table tasks * panel_stride]
    int panel_stride;
    int lt_begin, lt_end;    // level tasks of this launch
    int nb, maxb;            // matrices in this launch / slots of the table
    int items_per_task;
    int use_deps;
    int N;
    double* userD[MAX_BATCH];  // per slot: the caller's D
    long long ldD;
    int tma2d;               // 1: operand maps are 2-D {column, row} with one 16-column box per copy
    const short2* sym_tiles; // [items of a symmetric task] (tm, tn) of work item i: the tiles that touch the lower triangle, column-
                             // panel-major, or -- matrices that do not fit the L2 -- in bands of 16 column panels, row-major inside a
                             // band, so that the CTAs of a wave share a few A row blocks and B column panels
    const int* sym_panel_target;  // [tiles_n] completion count of a column panel of a symmetric task (DEP_PANEL_SYM)
    int* error_flag;         // set to 1 if a dependency wait exceeds the watchdog (never in a correct run)
    TraceRec* trace;         // nullable: per-item timeline, indexed by trace_base + work item of the launch
    int trace_base;
};

// BM x BN CTA tile, WM x WN warp tile (multiples of 16 / 8), BK k-rows per pipeline stage.
template <int BM_, int BN_, int WM_, int WN_, int BK_, int STAGES_, int MIN_CTAS_, int EARLYC_ = -1>
struct GemmCfg {
    static constexpr int BM = BM_, BN = BN_, WM = WM_, WN = WN_, BK = BK_, STAGES = STAGES_, MIN_CTAS = MIN_CTAS_;
    static constexpr int WARPS_M = BM / WM, WARPS_N = BN / WN;
    static constexpr int FM = WM / 8, FN = WN / 8;               // 8x8 DMMA fragments per warp tile
    static constexpr int CONSUMER_WARPS = WARPS_M * WARPS_N;
    static constexpr int CONSUMER_THREADS = CONSUMER_WARPS * 32;
    static constexpr int THREADS = CONSUMER_THREADS + 64;        // + producer warp + publisher warp
    static constexpr int SLAB_BYTES = BK * 128;                  // one 16-column slab: BK rows x 128 B
    // slabs per TMA box: the largest of 4, 2, 1 that divides both operand tiles (one tensor map serves both operands)
    static constexpr int BOX_SLABS = ((BM / 16) % 4 == 0 && (BN / 16) % 4 == 0) ? 4 : (((BM / 16) % 2 == 0 && (BN / 16) % 2 == 0) ? 2 : 1);
    static constexpr int BOX_BYTES = BOX_SLABS * SLAB_BYTES;
    static constexpr int A_BYTES = BM * BK * 8, B_BYTES = BN * BK * 8;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int BAR_OFFSET = STAGES * STAGE_BYTES;
    static constexpr int TRC_OFFSET = BAR_OFFSET + 256;          // [TILE_RING][4] u64 trace hand-off
    static constexpr int SMEM_BYTES = TRC_OFFSET + 64 + 1024;     // + alignment slack
    // small warp tiles have the registers to fetch the C tile as soon as the dependencies are known to be
    // satisfied (first full barrier), which takes one L2 round trip off the serial chain of the giant steps
    static constexpr bool EARLY_C = EARLYC_ < 0 ? (WM * WN <= 512) : (EARLYC_ != 0);
    static_assert(WM % 16 == 0 && WN % 8 == 0 && BM % WM == 0 && BN % WN == 0, "tile shapes");
    static_assert(WN % 16 == 0, "warp tiles are whole 16-column slabs");
    static_assert(BK % 8 == 0 && STAGES <= 8, "pipeline");
};

struct TileInfo {
    int task, tm, tn, stop;
    int item, pad;
    unsigned long long t_claim;
};

// Optional per-tile timeline (cheb_dm_set_trace): one record per work item, globaltimer nanoseconds.
struct TraceRec {
    int task, tm, tn, sm;
    unsigned long long t_claim;  // producer claimed the item
    unsigned long long t_desc;   // consumers received the descriptor (early dependencies satisfied)
    unsigned long long t_first;  // first operand stage landed (late dependencies satisfied, TMA round trip done)
    unsigned long long t_kend;   // K loop finished
    unsigned long long t_done;   // tile stored and published
};
__device__ __forceinline__ unsigned long long global_ns() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ int sm_id() {
    int v;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(v));
    return v;
}


// Producer-side wait for one dependency counter (global memory, written by red.release.gpu).
__device__ __forceinline__ void wait_counter(const int* ctr, int target, int* error_flag) {
    // Poll with relaxed loads (an acquire load invalidates the SM's L1 on every trip, under the consumer warps' feet),
    // then take the acquire once.
    if (ld_acquire_gpu(ctr) >= target) return;
    const long long t0 = clock64();
    while (ld_relaxed_gpu(ctr) < target) {
        if (clock64() - t0 > WATCHDOG_CLOCKS) {  // ~4 s: report instead of hanging
            atomicExch(error_flag, 1);
            break;
        }
    }
    (void)ld_acquire_gpu(ctr);
}

// Completion counters of a finished tile (after the gpu-scope fence): its column panel, the task, and -- symmetric task
// with BM a multiple of BN -- the column panel(s) its mirror lands in (the columns of the mirror are the rows of the tile).
template <int BM, int BN>
__device__ __forceinline__ void publish_tile(const LaunchArgs& args, const TileInfo& ti) {
    int* pd = args.panel_done + (size_t)ti.task * args.panel_stride;
    red_relaxed_gpu_add(pd + ti.tn, 1);
    if (BM % BN == 0 && args.tasks[ti.task].sym) {
        constexpr int R = (BM % BN == 0) ? BM / BN : 1;
        const int tiles_n = args.tasks[ti.task].tiles_n;
#pragma unroll
        for (int u = 0; u < R; ++u) {
            const int q = ti.tm * R + u;
            if (q != ti.tn && q < tiles_n) red_relaxed_gpu_add(pd + q, 1);
        }
    }
    red_relaxed_gpu_add(args.task_done + ti.task, 1);
}

template <class Cfg>
__global__ void __launch_bounds__(Cfg::THREADS, Cfg::MIN_CTAS) gemm_dmma_kernel(const LaunchArgs args) {
    constexpr int BM = Cfg::BM, BN = Cfg::BN, BK = Cfg::BK, STAGES = Cfg::STAGES;
    constexpr int FM = Cfg::FM, FN = Cfg::FN;
    constexpr int SLAB_BYTES = Cfg::SLAB_BYTES;
    extern __shared__ uint8_t smem_raw[];
    // 1024-byte alignment: the 128B swizzle pattern is a function of address bits [7:9]
    // (the pad is applied as an offset so that the pointer keeps its shared address space: LDS, not generic LD)
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Cfg::BAR_OFFSET);
    // bars[0..S) full, [S..2S) empty, [2S..2S+R) tile_full, [2S+R..2S+2R) tile_empty, [2S+2R..2S+3R) tile stored
    TileInfo* ring = reinterpret_cast<TileInfo*>(smem + Cfg::BAR_OFFSET + 192);
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t bar_base = smem_u32(bars);
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + s); };
    auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + TILE_RING + s); };
    // one "stored" barrier per descriptor slot: a consumer warp may run one tile ahead of a slow warp (next tile's K
    // loop fits the free ring, or epilogue-only tiles), and its arrive for tile n+1 must not complete tile n's phase
    auto stored_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + 2 * TILE_RING + s); };
    unsigned long long* trc = reinterpret_cast<unsigned long long*>(smem + Cfg::TRC_OFFSET);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), Cfg::CONSUMER_WARPS);
        }
        for (int s = 0; s < TILE_RING; ++s) {
            mbar_init(tfull_bar(s), 1);
            mbar_init(tempty_bar(s), Cfg::CONSUMER_WARPS + 1);  // consumer warps + publisher
            mbar_init(stored_bar(s), Cfg::CONSUMER_WARPS);
        }
        fence_mbar_init();
    }
    __syncthreads();

    const int ipt = args.items_per_task;
    const int item_end = (args.lt_end - args.lt_begin) * args.nb * ipt;

    if (warp == Cfg::CONSUMER_WARPS) {
        // =================================== producer warp ===================================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            int tslot = 0;
            uint32_t tphase = 0;
            const int tbase = args.lt_begin * args.maxb;   // first table task of this launch
            unsigned long long done_tasks[8] = {0ull, 0ull, 0ull, 0ull, 0ull, 0ull, 0ull, 0ull};  // "task complete" seen (rel. index < 512)
            unsigned long long fenced_maps[4] = {0ull, 0ull, 0ull, 0ull};  // tensor maps this CTA has acquired
            auto acquire_map = [&](int m) {
                if (m < 256 && ((fenced_maps[m >> 6] >> (m & 63)) & 1ull)) return;
                fence_tensormap_acquire(args.maps + m);
                if (m < 256) fenced_maps[m >> 6] |= 1ull << (m & 63);
            };
            // One dependency of task `tk` for column panel `tn` (no-op when already observed complete).
            auto wait_dep = [&](const Task* tk, int d, int tn) {
                const int kind = tk->dep_kind[d], idx = tk->dep_idx[d], target = tk->dep_target[d];
                const int rel = idx - tbase;
                const int* ctr;
                int tgt = target;
                if (kind == DEP_TASK) {
                    if (rel >= 0 && rel < 512 && ((done_tasks[rel >> 6] >> (rel & 63)) & 1ull)) return;
                    ctr = args.task_done + idx;
                } else {
                    ctr = args.panel_done + (size_t)idx * args.panel_stride + tn;
                    if (kind == DEP_PANEL_SYM) tgt = __ldg(args.sym_panel_target + tn);
                }
                wait_counter(ctr, tgt, args.error_flag);
                if (kind == DEP_TASK && rel >= 0 && rel < 512) done_tasks[rel >> 6] |= 1ull << (rel & 63);
            };
            for (;;) {
                const int item = atomicAdd(args.work_counter, 1);
                const bool stop = item >= item_end;
                const unsigned long long t_claim = args.trace ? global_ns() : 0ull;
                int tm = 0, tn = 0, cur = tbase;
                const Task* tk = nullptr;
                if (!stop) {
                    const int tq = item / ipt, local = item - tq * ipt;
                    const int lt = tq / args.nb, slot = tq - lt * args.nb;
                    cur = (args.lt_begin + lt) * args.maxb + slot;
                    tk = args.tasks + cur;
                    const int tiles_m = tk->tiles_m;
                    if (!tk->sym) {
                        tn = local / tiles_m;  // column-panel-major order: a panel's tiles are consecutive
                        tm = local - tn * tiles_m;
                    } else {
                        // symmetric task: the plan's item -> tile table (lower-triangle tiles in raster order)
                        const short2 tt = __ldg(args.sym_tiles + local);
                        tm = tt.x;
                        tn = tt.y;
                    }
                    // early dependencies: operands of the low-order sum, which the consumers read before the K loop
                    if (args.use_deps)
                        for (int d = 0; d < tk->ndeps_early; ++d) wait_dep(tk, d, tn);
                }
                // publish the tile descriptor to the consumer warps (mbarrier arrive = release, CTA scope)
                mbar_wait(tempty_bar(tslot), tphase ^ 1);
                ring[tslot].task = cur;
                ring[tslot].tm = tm;
                ring[tslot].tn = tn;
                ring[tslot].stop = stop ? 1 : 0;
                ring[tslot].item = item;
                ring[tslot].t_claim = t_claim;
                mbar_arrive(tfull_bar(tslot));
                if (++tslot == TILE_RING) { tslot = 0; tphase ^= 1; }
                if (stop) break;

                // late dependencies: the TMA operands and the C tile
                if (args.use_deps) {
                    const int nd = tk->ndeps;
                    for (int d = tk->ndeps_early; d < nd; ++d) wait_dep(tk, d, tn);
                    fence_proxy_async_global();  // data written through the generic proxy, read next by TMA
                }
                const int ktiles = tk->ktiles;
                const int kchunks = ktiles > 0 ? tk->kchunks : 0;
                for (int kc = 0; kc < kchunks; ++kc) {
                    const CUtensorMap* mapA = args.maps + tk->mapA + kc;
                    const CUtensorMap* mapB = args.maps + tk->mapB + kc;
                    acquire_map(tk->mapA + kc);
                    acquire_map(tk->mapB + kc);
                    const int slabA = tm * (BM / 16), slabB = tn * (BN / 16);
                    for (int kt = 0; kt < ktiles; ++kt) {
                        mbar_wait(empty_bar(stage), phase ^ 1);
                        const uint32_t sA = smem_base + stage * Cfg::STAGE_BYTES;
                        const uint32_t sB = sA + Cfg::A_BYTES;
                        mbar_arrive_expect_tx(full_bar(stage), Cfg::STAGE_BYTES);
                        if (!args.tma2d) {
#pragma unroll
                            for (int b = 0; b < BM / (16 * Cfg::BOX_SLABS); ++b)
                                tma_load_3d(sA + b * Cfg::BOX_BYTES, mapA, full_bar(stage), 0, kt * BK, slabA + Cfg::BOX_SLABS * b);
#pragma unroll
                            for (int b = 0; b < BN / (16 * Cfg::BOX_SLABS); ++b)
                                tma_load_3d(sB + b * Cfg::BOX_BYTES, mapB, full_bar(stage), 0, kt * BK, slabB + Cfg::BOX_SLABS * b);
                        } else {
#pragma unroll
                            for (int b = 0; b < BM / 16; ++b)
                                tma_load_2d(sA + b * SLAB_BYTES, mapA, full_bar(stage), (slabA + b) * 16, kt * BK);
#pragma unroll
                            for (int b = 0; b < BN / 16; ++b)
                                tma_load_2d(sB + b * SLAB_BYTES, mapB, full_bar(stage), (slabB + b) * 16, kt * BK);
                        }
                        if (++stage == STAGES) { stage = 0; phase ^= 1; }
                    }
                }
            }
        }
        return;
    }

    if (warp == Cfg::CONSUMER_WARPS + 1) {
        // =================================== publisher warp ===================================
        // Publishes the completion of each tile: waits until every consumer warp has stored its part (mbarrier
        // arrive = release, CTA scope), makes the tile visible device-wide with ONE gpu-scope fence (cumulative over
        // the stores it has synchronised with), then bumps the two counters.  The consumer warps meanwhile go
        // straight on to their next tile.  Waiting producers pair this with ld.acquire.gpu + fence.proxy.async.
        // The descriptor slot is released only after publication, so the consumers are never two tiles ahead; each
        // descriptor slot has its own "stored" barrier, so being ONE tile ahead cannot be mis-attributed either.
        if (lane == 0) {
            int tslot = 0;
            uint32_t tphase = 0;
            for (;;) {
                mbar_wait(tfull_bar(tslot), tphase);
                const TileInfo ti = ring[tslot];
                if (!ti.stop) {
                    mbar_wait(stored_bar(tslot), tphase);  // slot s is used once per ring cycle: same phase as its descriptor
                    fence_acq_rel_gpu();
                    publish_tile<BM, BN>(args, ti);
                    if (args.trace != nullptr) {
                        TraceRec r;
                        r.task = ti.task; r.tm = ti.tm; r.tn = ti.tn; r.sm = sm_id();
                        r.t_claim = ti.t_claim; r.t_desc = trc[tslot * 4 + 0]; r.t_first = trc[tslot * 4 + 1];
                        r.t_kend = trc[tslot * 4 + 2]; r.t_done = global_ns();
                        args.trace[args.trace_base + ti.item] = r;
                    }
                }
                mbar_arrive_dep(tempty_bar(tslot), ti.task ^ ti.tm ^ ti.tn ^ ti.stop ^ ti.item ^ (int)ti.t_claim);
                if (ti.stop) break;
                if (++tslot == TILE_RING) { tslot = 0; tphase ^= 1; }
            }
        }
        return;
    }

    // ======================================= consumer warps =======================================
    const int wm = warp / Cfg::WARPS_N, wn = warp % Cfg::WARPS_N;
    const int g = lane >> 2, t = lane & 3;
    // Per-lane fragment offsets inside a stage (see header comment).  For k4-step j: jh = j>>1, par = j&1,
    // physical k-row r = 8*jh + par + 2t.  Column c = w*W + i*8 + g of the operand tile lives in slab c>>4,
    // 16-byte chunk ((c&15)>>1) ^ (r&7), half c&1.
    uint32_t aoff[2], boff[2];
#pragma unroll
    for (int par = 0; par < 2; ++par) {
        const uint32_t x = par + 2 * t;
        const uint32_t lo = x * 128 + ((((uint32_t)g >> 1) ^ x) << 4) + (g & 1) * 8;
        aoff[par] = (wm * (Cfg::WM / 16)) * SLAB_BYTES + lo;
        boff[par] = Cfg::A_BYTES + (wn * (Cfg::WN / 16)) * SLAB_BYTES + lo;
    }

    int stage = 0;
    uint32_t phase = 0;
    int tslot = 0;
    uint32_t tphase = 0;
    const int N = args.N;

    for (;;) {
        mbar_wait(tfull_bar(tslot), tphase);
        const TileInfo ti = ring[tslot];
        const int ti_slot = tslot;
        // every lane must hold its copy of the descriptor before the slot is handed back (the arrive is tied to the
        // loaded values; __syncwarp orders the other lanes' loads before lane 0's arrive)
        const int ti_dep = ti.task ^ ti.tm ^ ti.tn ^ ti.stop ^ ti.item ^ (int)ti.t_claim ^ (int)(ti.t_claim >> 32);
        const int ti_dep_all = (int)__reduce_xor_sync(0xffffffffu, (unsigned)ti_dep);  // needs every lane's copy
        if (lane == 0) mbar_arrive_dep(tempty_bar(tslot), ti_dep_all);
        if (++tslot == TILE_RING) { tslot = 0; tphase ^= 1; }
        if (ti.stop) break;
        const Task* tk = args.tasks + ti.task;
        const bool tracing = (args.trace != nullptr) && threadIdx.x == 0;
        unsigned long long t_desc = 0, t_first = 0, t_kend = 0;
        if (tracing) t_desc = global_ns();
        const int row0 = ti.tm * BM + wm * Cfg::WM + g;
        const int col0 = ti.tn * BN + wn * Cfg::WN + 2 * t;

        double acc[FM][FN][2];
#pragma unroll
        for (int i = 0; i < FM; ++i)
#pragma unroll
            for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

        // ---- prologue: low-order sum  sum_i coef_i T_i  (Eq. 21).  Small warp tiles have the registers to form
        // it BEFORE the K loop (its operands are guarded by the task's early dependencies, which the producer checked
        // before publishing this tile), so the work overlaps the wait for the previous giant step instead of extending
        // the serial chain.  It is kept in registers of its own and added in the epilogue: starting the accumulator
        // from it would make every DMMA rounding relative to the (large) sum instead of the (small) running product
        // and measurably costs accuracy (cfg4: |dtr D| 7e-10 -> 3e-9).  Large warp tiles form it in the epilogue.
        constexpr bool PRE_SUM = (FM * FN <= 4) || (FM * FN <= 8 && Cfg::THREADS <= 320);  // 18-warp CTAs have 96 registers per thread
        constexpr int PRE_U = (FM * FN <= 4) ? 4 : 2;  // operands in flight per iteration (register budget)
        double pre[PRE_SUM ? FM : 1][PRE_SUM ? FN : 1][2];
#pragma unroll
        for (int i = 0; i < (PRE_SUM ? FM : 1); ++i)
#pragma unroll
            for (int j = 0; j < (PRE_SUM ? FN : 1); ++j) pre[i][j][0] = pre[i][j][1] = 0.0;
        const int ns = tk->sum_count;
        if (PRE_SUM && ns > 0) {
            const double* coef = tk->coef;
            const long long lds = tk->lds, sstride = tk->sum_stride;
            const double* sb = tk->sum_base + (long long)row0 * lds + col0;
            int s = 0;
            for (; s + PRE_U - 1 < ns; s += PRE_U) {  // PRE_U operands in flight per iteration
                double w[PRE_U];
                double2 v[PRE_U][PRE_SUM ? FM : 1][PRE_SUM ? FN : 1];
#pragma unroll
                for (int u = 0; u < PRE_U; ++u) {
                    w[u] = __ldg(coef + s + u);
                    const double* pu = sb + (long long)(s + u) * sstride;
#pragma unroll
                    for (int i = 0; i < (PRE_SUM ? FM : 1); ++i)
#pragma unroll
                        for (int j = 0; j < (PRE_SUM ? FN : 1); ++j) {
                            const bool in = (row0 + i * 8 < N) && (col0 + j * 8 < N);  // pad column N (odd N) holds zeros
                            v[u][i][j] = in ? __ldcg(reinterpret_cast<const double2*>(pu + (long long)(i * 8) * lds + j * 8)) : make_double2(0.0, 0.0);
                        }
                }
#pragma unroll
                for (int u = 0; u < PRE_U; ++u)
#pragma unroll
                    for (int i = 0; i < (PRE_SUM ? FM : 1); ++i)
#pragma unroll
                        for (int j = 0; j < (PRE_SUM ? FN : 1); ++j) {
                            pre[i][j][0] = fma(w[u], v[u][i][j].x, pre[i][j][0]);
                            pre[i][j][1] = fma(w[u], v[u][i][j].y, pre[i][j][1]);
                        }
            }
            for (; s < ns; ++s) {
                const double w0 = __ldg(coef + s);
                const double* p0 = sb + (long long)s * sstride;
#pragma unroll
                for (int i = 0; i < (PRE_SUM ? FM : 1); ++i)
#pragma unroll
                    for (int j = 0; j < (PRE_SUM ? FN : 1); ++j)
                        if ((row0 + i * 8 < N) && (col0 + j * 8 < N)) {
                            const double2 v = __ldcg(reinterpret_cast<const double2*>(p0 + (long long)(i * 8) * lds + j * 8));
                            pre[i][j][0] = fma(w0, v.x, pre[i][j][0]);
                            pre[i][j][1] = fma(w0, v.y, pre[i][j][1]);
                        }
            }
        }

        // ---- C tile: fetched as soon as the first full barrier shows that the late dependencies hold ----
        const double* Cp = tk->C;
        const long long ldc = tk->ldc;
        const bool cvec = ((ldc & 1) == 0) && ((reinterpret_cast<uintptr_t>(Cp) & 15) == 0);
        double creg[Cfg::EARLY_C ? FM : 1][Cfg::EARLY_C ? FN : 1][2];
        auto load_c = [&](int i, int j, double& c0, double& c1) {
            const int r = row0 + i * 8, c = col0 + j * 8;
            c0 = 0.0;
            c1 = 0.0;
            if (r < N && c < N) {
                const double* p = Cp + (long long)r * ldc + c;
                if (cvec && c + 1 < N) {
                    const double2 v = __ldcg(reinterpret_cast<const double2*>(p));
                    c0 = v.x;
                    c1 = v.y;
                } else {
                    c0 = __ldcg(p);
                    if (c + 1 < N) c1 = __ldcg(p + 1);
                }
            }
        };
        bool c_loaded = false;

        // A stage is handed back to the producer one iteration late: when the NEXT stage's full barrier has been
        // passed, every DMMA of the previous iteration has issued, hence every ld.shared feeding them has returned.
        // (Arriving at the end of the same iteration is not safe: the arrive can overtake loads still in flight and
        // the producer's next TMA write then races with them.)
        const int ktiles = tk->ktiles * (tk->ktiles > 0 ? tk->kchunks : 0);
        int prev_stage = -1;
        for (int kt = 0; kt < ktiles; ++kt) {
            mbar_wait(full_bar(stage), phase);
            if (tracing && kt == 0) t_first = global_ns();
            if (Cfg::EARLY_C && kt == 0 && Cp != nullptr) {
#pragma unroll
                for (int i = 0; i < FM; ++i)
#pragma unroll
                    for (int j = 0; j < FN; ++j) load_c(i, j, creg[Cfg::EARLY_C ? i : 0][Cfg::EARLY_C ? j : 0][0], creg[Cfg::EARLY_C ? i : 0][Cfg::EARLY_C ? j : 0][1]);
                c_loaded = true;
            }
            const uint8_t* sbase = smem + stage * Cfg::STAGE_BYTES;
#pragma unroll
            for (int j = 0; j < BK / 4; ++j) {
                const int jh = j >> 1, par = j & 1;
                double a[FM], b[FN];
#pragma unroll
                for (int i = 0; i < FM; ++i)
                    a[i] = *reinterpret_cast<const double*>(sbase + ((aoff[par] ^ ((i & 1) << 6)) + (i >> 1) * SLAB_BYTES + jh * 1024));
#pragma unroll
                for (int i = 0; i < FN; ++i)
                    b[i] = *reinterpret_cast<const double*>(sbase + ((boff[par] ^ ((i & 1) << 6)) + (i >> 1) * SLAB_BYTES + jh * 1024));
                if (j == 0 && prev_stage >= 0) {  // previous stage back to the producer (after this stage's barrier, off the
                    __syncwarp();                 // path from the barrier to the first loads)
                    if (lane == 0) mbar_arrive(empty_bar(prev_stage));
                }
#pragma unroll
                for (int im = 0; im < FM; ++im)
#pragma unroll
                    for (int jn = 0; jn < FN; ++jn) dmma_884(acc[im][jn][0], acc[im][jn][1], a[im], b[jn]);
            }
            prev_stage = stage;
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        if (prev_stage >= 0) {
            // last stage of the tile: the loop-exit branch separates the arrive from the DMMAs that consumed the loads
            __syncwarp();
            int dep = 0;
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dep ^= __double2hiint(acc[i][j][0]) ^ __double2hiint(acc[i][j][1]);
            if (lane == 0) mbar_arrive_dep(empty_bar(prev_stage), dep);
        }

        // ------------------------------------ epilogue ------------------------------------
        if (tracing) t_kend = global_ns();
        const double alpha = tk->alpha;
#pragma unroll
        for (int i = 0; i < FM; ++i)
#pragma unroll
            for (int j = 0; j < FN; ++j) {
                acc[i][j][0] *= alpha;
                acc[i][j][1] *= alpha;
            }
        if (Cp != nullptr) {
            const double beta = tk->beta;
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) {
                    double c0, c1;
                    if (Cfg::EARLY_C && c_loaded) {
                        c0 = creg[Cfg::EARLY_C ? i : 0][Cfg::EARLY_C ? j : 0][0];
                        c1 = creg[Cfg::EARLY_C ? i : 0][Cfg::EARLY_C ? j : 0][1];
                    } else {
                        load_c(i, j, c0, c1);
                    }
                    acc[i][j][0] = fma(beta, c0, acc[i][j][0]);
                    acc[i][j][1] = fma(beta, c1, acc[i][j][1]);
                }
        }
        if (ns > 0) {
            if (PRE_SUM) {
#pragma unroll
                for (int i = 0; i < (PRE_SUM ? FM : 1); ++i)
#pragma unroll
                    for (int j = 0; j < (PRE_SUM ? FN : 1); ++j) {
                        acc[PRE_SUM ? i : 0][PRE_SUM ? j : 0][0] += pre[i][j][0];
                        acc[PRE_SUM ? i : 0][PRE_SUM ? j : 0][1] += pre[i][j][1];
                    }
            } else {
                // workspace matrices: even ld, 16-byte aligned rows, zero pad columns
                const double* coef = tk->coef;
                const long long lds = tk->lds, sstride = tk->sum_stride;
                const double* sb = tk->sum_base + (long long)row0 * lds + col0;
                for (int s = 0; s < ns; ++s) {
                    const double w = __ldg(coef + s);
                    const double* ps = sb + (long long)s * sstride;
#pragma unroll
                    for (int i = 0; i < FM; ++i)
#pragma unroll
                        for (int j = 0; j < FN; ++j)
                            if ((row0 + i * 8 < N) && (col0 + j * 8 < N)) {
                                const double2 v = __ldcg(reinterpret_cast<const double2*>(ps + (long long)(i * 8) * lds + j * 8));
                                acc[i][j][0] = fma(w, v.x, acc[i][j][0]);
                                acc[i][j][1] = fma(w, v.y, acc[i][j][1]);
                            }
                }
            }
        }
        {
            double diag = tk->diag_const;
            if (tk->diag_ptr != nullptr) diag += __ldg(tk->diag_ptr);
            if (diag != 0.0) {
#pragma unroll
                for (int i = 0; i < FM; ++i)
#pragma unroll
                    for (int j = 0; j < FN; ++j) {
                        const int r = row0 + i * 8, c = col0 + j * 8;
                        if (r == c) acc[i][j][0] += diag;
                        if (r == c + 1) acc[i][j][1] += diag;
                    }
            }
        }
        {
            double* Out = tk->out_is_user ? args.userD[tk->slot] : tk->Out;
            const long long ldo = tk->out_is_user ? args.ldD : tk->ldo;
            const bool vec = ((ldo & 1) == 0) && ((reinterpret_cast<uintptr_t>(Out) & 15) == 0);
#pragma unroll
            for (int i = 0; i < FM; ++i) {
                const int r = row0 + i * 8;
#pragma unroll
                for (int j = 0; j < FN; ++j) {
                    const int c = col0 + j * 8;
                    if (r < N && c < N) {
                        double* p = Out + (long long)r * ldo + c;
                        if (vec && c + 1 < N) {
                            __stcg(reinterpret_cast<double2*>(p), make_double2(acc[i][j][0], acc[i][j][1]));
                        } else {
                            __stcg(p, acc[i][j][0]);
                            if (c + 1 < N) __stcg(p + 1, acc[i][j][1]);
                        }
                    }
                }
            }
            if (tk->sym) {
                // Mirror: an 8x8 block whose transposed position falls into a tile that is not a work item (tile
                // (tm', tn') with tm' BM + BM - 1 < tn' BN, i.e. strictly above the diagonal) is transposed inside the
                // warp with shuffles and stored there, row-contiguous like the direct store.  Lane (g, t) of the
                // transposed block holds C[2t][g], C[2t+1][g], which live in lanes (2t, g>>1) and (2t+1, g>>1).
                const int src0 = (2 * t) * 4 + (g >> 1), src1 = src0 + 4;
#pragma unroll
                for (int i = 0; i < FM; ++i) {
                    const int R0 = ti.tm * BM + wm * Cfg::WM + i * 8;  // rows of the block
#pragma unroll
                    for (int j = 0; j < FN; ++j) {
                        const int C0 = ti.tn * BN + wn * Cfg::WN + j * 8;  // columns of the block
                        if ((C0 / BM) * BM + BM - 1 < (R0 / BN) * BN) {   // warp-uniform
                            const double a0 = __shfl_sync(0xffffffffu, acc[i][j][0], src0), a1 = __shfl_sync(0xffffffffu, acc[i][j][1], src0);
                            const double b0 = __shfl_sync(0xffffffffu, acc[i][j][0], src1), b1 = __shfl_sync(0xffffffffu, acc[i][j][1], src1);
                            const double w0 = (g & 1) ? a1 : a0, w1 = (g & 1) ? b1 : b0;
                            const int rr = C0 + g, cc = R0 + 2 * t;  // transposed position: row C0+g, columns R0+2t, R0+2t+1
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
                }
            }
        }
        // --------------------- hand the tile over to the publisher warp ---------------------
        if (tracing) {
            trc[ti_slot * 4 + 0] = t_desc;
            trc[ti_slot * 4 + 1] = t_first;
            trc[ti_slot * 4 + 2] = t_kend;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(stored_bar(ti_slot));
    }
}

}  // namespace chebdm
