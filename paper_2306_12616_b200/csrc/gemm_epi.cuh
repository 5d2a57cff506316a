// gemm_epi.cuh -- persistent grouped FP64 GEMM with SPECIALISED EPILOGUE WARPS, for the small tiles of small N.
//
// Same tasks, work queue, dependency counters and operand pipeline as gemm_dmma.cuh (one task = one product
//     Out = alpha * (A^T B) + beta * C + sum_i coef_i S_i + diag * I
// of the recurrence: Eq. 7 / 22-23 / Alg. 1, Eq. 4 and its Clenshaw form, Eq. 21), but
// the consumer warps only run the K loop: when a tile's K loop ends they park their accumulators in a shared-memory
// staging tile and go straight on to the next work item, while four epilogue warps -- which fetched the C tile and
// the low-order sum of the SAME item from L2 during its K loop -- combine, store the tile, mirror it (symmetric-tile
// skipping) and publish its completion.  At N ~ 500 the epilogue of a 64 x 32 tile (C and G loads, stores, mirror,
// gpu-scope fence) is 1.7-3.5 us against a 9-18 us K loop; here it overlaps the next item's K loop, and with two
// waves of items per level the publish -> poll -> TMA latency of a giant step hides under the other wave as well.
// (The paper overlaps with streams, and pays separate passes for the additions.)
//
// Warp roles (16 warps, 128 registers per thread): 0..7 consumers, 8 producer (one lane: work queue, dependency
// waits, TMA), 9..11 exit at once, 12..15 epilogue.  A 64 x 32 tile is computed by 2 k-halves x (2 x 2 warps of
// 32 x 16): the halves are added by the epilogue warps when they read the staging tile.
//
// The staging tile is row-major with a row pitch of BN + 8 doubles (pitch = 64 mod 128 bytes: the consumers' 8-row
// fragment stores and the epilogue's row reads are conflict-free); the mirror reads it back by columns of 4-row quads
// (lanes along a row: conflict-free) and stores whole 32-byte sectors.
#pragma once
#include "gemm_dmma.cuh"

namespace chebdm {

template <int BM_, int BN_, int WM_, int WN_, int KSPLIT_, int BK_, int STAGES_>
struct EpiCfg {
    static constexpr int BM = BM_, BN = BN_, WM = WM_, WN = WN_, KSPLIT = KSPLIT_, BK = BK_, STAGES = STAGES_;
    static constexpr int WARPS_M = BM / WM, WARPS_N = BN / WN;
    static constexpr int FM = WM / 8, FN = WN / 8;
    static constexpr int CONSUMER_WARPS = KSPLIT * WARPS_M * WARPS_N;
    static constexpr int PRODUCER_WARP = CONSUMER_WARPS;
    static constexpr int EPI_WARP0 = 12, EPI_WARPS = 4, EPI_THREADS = EPI_WARPS * 32;
    static constexpr int THREADS = 512;
    static constexpr int RING = 4;                               // tile descriptors in flight (producer, consumers, epilogue)
    static constexpr int SLAB_BYTES = BK * 128;
    static constexpr int BOX_SLABS = ((BM / 16) % 4 == 0 && (BN / 16) % 4 == 0) ? 4 : (((BM / 16) % 2 == 0 && (BN / 16) % 2 == 0) ? 2 : 1);
    static constexpr int BOX_BYTES = BOX_SLABS * SLAB_BYTES;
    static constexpr int A_BYTES = BM * BK * 8, B_BYTES = BN * BK * 8;
    static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
    static constexpr int STG_LD = BN + 8;                        // doubles per staging row
    static constexpr int STG_HALF = BM * STG_LD;                 // doubles per k-half
    static constexpr int STG_OFFSET = STAGES * STAGE_BYTES;
    static constexpr int STG_BYTES = KSPLIT * STG_HALF * 8;
    static constexpr int BAR_OFFSET = STG_OFFSET + STG_BYTES;    // mbarriers (<= 256 B), then the descriptor ring, then trace words
    static constexpr int RING_OFFSET = BAR_OFFSET + 256;
    static constexpr int TRC_OFFSET = RING_OFFSET + RING * 32;
    static constexpr int SMEM_BYTES = TRC_OFFSET + RING * 32 + 1024;
    static constexpr int K4_PER_HALF = BK / 4 / KSPLIT;          // k4-steps of one stage per k-half
    static constexpr int CP = BN / 2;                            // double2 columns of a tile row
    static constexpr int ROWS_PER_PASS = EPI_THREADS / CP;       // rows the epilogue warps cover per pass
    static constexpr int NPASS = BM / ROWS_PER_PASS;
    static_assert(CONSUMER_WARPS == 8, "eight consumer warps");
    static_assert(WM % 16 == 0 && WN % 16 == 0 && BM % WM == 0 && BN % WN == 0, "tile shapes");
    static_assert((BK / 4) % (2 * KSPLIT) == 0 && STAGES <= 8, "pipeline");
    static_assert((BN * 8) % 128 == 0 && BM % 32 == 0 && BN % 32 == 0 && BN <= BM, "staging layout");
    static_assert(2 * STAGES + 4 * RING + 2 <= 32, "barrier block");
    static_assert(sizeof(TileInfo) == 32, "descriptor size");
};

template <class Cfg>
__global__ void __launch_bounds__(Cfg::THREADS, 1) gemm_epi_kernel(const LaunchArgs args) {
    constexpr int BM = Cfg::BM, BN = Cfg::BN, BK = Cfg::BK, STAGES = Cfg::STAGES, RING = Cfg::RING;
    constexpr int FM = Cfg::FM, FN = Cfg::FN;
    constexpr int SLAB_BYTES = Cfg::SLAB_BYTES;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    double* stg = reinterpret_cast<double*>(smem + Cfg::STG_OFFSET);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Cfg::BAR_OFFSET);
    TileInfo* ring = reinterpret_cast<TileInfo*>(smem + Cfg::RING_OFFSET);
    unsigned long long* trc = reinterpret_cast<unsigned long long*>(smem + Cfg::TRC_OFFSET);
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t bar_base = smem_u32(bars);
    // [0,S) full | [S,2S) empty | [2S,2S+R) tile_full | [..+R) tile_empty | [..+R) deps_ok | [..+R) epi_done | acc_full | acc_empty
    // (epi_done is per descriptor slot: an epilogue warp may run one product-free item ahead of a slow one, and its arrive
    // for item n+1 must not complete item n's phase)
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + s); };
    auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + RING + s); };
    auto deps_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + 2 * RING + s); };
    auto epidone_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + 3 * RING + s); };
    const uint32_t accfull_bar = bar_base + 8u * (2 * STAGES + 4 * RING);
    const uint32_t accempty_bar = accfull_bar + 8u;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), Cfg::CONSUMER_WARPS / Cfg::KSPLIT);  // the warps that read the stage (see the K loop)
        }
        for (int s = 0; s < RING; ++s) {
            mbar_init(tfull_bar(s), 1);
            mbar_init(tempty_bar(s), Cfg::CONSUMER_WARPS + 1);  // consumer warps + the epilogue leader
            mbar_init(deps_bar(s), 1);
            mbar_init(epidone_bar(s), Cfg::EPI_WARPS);
        }
        mbar_init(accfull_bar, Cfg::CONSUMER_WARPS);
        mbar_init(accempty_bar, Cfg::EPI_WARPS);
        fence_mbar_init();
    }
    __syncthreads();

    const int ipt = args.items_per_task;
    const int item_end = (args.lt_end - args.lt_begin) * args.nb * ipt;
    const int N = args.N;

    if (warp == Cfg::PRODUCER_WARP) {
        // =================================== producer warp ===================================
        if (lane != 0) return;
        int stage = 0;
        uint32_t phase = 0;
        int tslot = 0;
        uint32_t tphase = 0;
        const int tbase = args.lt_begin * args.maxb;
        unsigned long long done_tasks[8] = {0ull, 0ull, 0ull, 0ull, 0ull, 0ull, 0ull, 0ull};
        unsigned long long fenced_maps[4] = {0ull, 0ull, 0ull, 0ull};
        auto acquire_map = [&](int m) {
            if (m < 256 && ((fenced_maps[m >> 6] >> (m & 63)) & 1ull)) return;
            fence_tensormap_acquire(args.maps + m);
            if (m < 256) fenced_maps[m >> 6] |= 1ull << (m & 63);
        };
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
                    tn = local / tiles_m;
                    tm = local - tn * tiles_m;
                } else {
                    const short2 tt = __ldg(args.sym_tiles + local);  // the plan's item -> tile table (raster order)
                    tm = tt.x;
                    tn = tt.y;
                }
                if (args.use_deps)
                    for (int d = 0; d < tk->ndeps_early; ++d) wait_dep(tk, d, tn);
            }
            mbar_wait(tempty_bar(tslot), tphase ^ 1);
            ring[tslot].task = cur;
            ring[tslot].tm = tm;
            ring[tslot].tn = tn;
            ring[tslot].stop = stop ? 1 : 0;
            ring[tslot].item = item;
            ring[tslot].t_claim = t_claim;
            mbar_arrive(tfull_bar(tslot));
            const uint32_t my_deps = deps_bar(tslot);
            if (++tslot == RING) { tslot = 0; tphase ^= 1; }
            if (stop) break;

            if (args.use_deps) {
                const int nd = tk->ndeps;
                for (int d = tk->ndeps_early; d < nd; ++d) wait_dep(tk, d, tn);
                fence_proxy_async_global();
            }
            mbar_arrive(my_deps);  // the epilogue warps may fetch this item's C tile now (release, CTA scope)
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
                        for (int b = 0; b < BM / 16; ++b) tma_load_2d(sA + b * SLAB_BYTES, mapA, full_bar(stage), (slabA + b) * 16, kt * BK);
#pragma unroll
                        for (int b = 0; b < BN / 16; ++b) tma_load_2d(sB + b * SLAB_BYTES, mapB, full_bar(stage), (slabB + b) * 16, kt * BK);
                    }
                    if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
        return;
    }

    if (warp >= Cfg::EPI_WARP0) {
        // =================================== epilogue warps ===================================
        const int et = threadIdx.x - Cfg::EPI_WARP0 * 32;           // 0..127
        const int cp = et % Cfg::CP, rg = et / Cfg::CP;             // double2 column, row inside a pass
        const bool leader = (et == 0);
        int tslot = 0;
        uint32_t tphase = 0, aphase = 0;
        for (;;) {
            mbar_wait(tfull_bar(tslot), tphase);
            const TileInfo ti = ring[tslot];
            const int my_slot = tslot;
            const uint32_t my_phase = tphase;
            if (++tslot == RING) { tslot = 0; tphase ^= 1; }
            if (ti.stop) {
                __syncwarp();
                if (leader) mbar_arrive(tempty_bar(my_slot));
                break;
            }
            const Task* tk = args.tasks + ti.task;
            const int row_t = ti.tm * BM, col_t = ti.tn * BN;
            const int col = col_t + 2 * cp;
            double* Out = tk->out_is_user ? args.userD[tk->slot] : tk->Out;
            const long long ldo = tk->out_is_user ? args.ldD : tk->ldo;
            const bool vec = ((ldo & 1) == 0) && ((reinterpret_cast<uintptr_t>(Out) & 15) == 0);

            // e = beta C + sum_i coef_i S_i + diag I, gathered while the consumers run this item's K loop
            double2 e[Cfg::NPASS];
#pragma unroll
            for (int i = 0; i < Cfg::NPASS; ++i) e[i] = make_double2(0.0, 0.0);
            const int ns = tk->sum_count;
            if (ns > 0) {  // workspace matrices: even ld, 16-byte aligned rows, zero pad columns; guarded by early deps
                const double* coef = tk->coef;
                const long long lds = tk->lds, sstride = tk->sum_stride;
                const double* sb = tk->sum_base + (long long)(row_t + rg) * lds + col;
                constexpr int U = (Cfg::NPASS <= 8) ? 2 : 1;  // operands in flight (register budget: 128 per thread)
                for (int s = 0; s < ns; s += U) {
                    double w[U];
                    double2 v[U][Cfg::NPASS];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        const bool live = (s + u < ns);
                        w[u] = live ? __ldg(coef + s + u) : 0.0;
#pragma unroll
                        for (int i = 0; i < Cfg::NPASS; ++i) {
                            const int r = row_t + rg + i * Cfg::ROWS_PER_PASS;
                            const bool in = live && (r < N) && (col < N);
                            const double* p0 = sb + (long long)(s + u) * sstride + (long long)(i * Cfg::ROWS_PER_PASS) * lds;
                            v[u][i] = in ? __ldcg(reinterpret_cast<const double2*>(p0)) : make_double2(0.0, 0.0);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u)
#pragma unroll
                        for (int i = 0; i < Cfg::NPASS; ++i) {
                            e[i].x = fma(w[u], v[u][i].x, e[i].x);
                            e[i].y = fma(w[u], v[u][i].y, e[i].y);
                        }
                }
            }
            {
                double diag = tk->diag_const;
                if (tk->diag_ptr != nullptr) diag += __ldg(tk->diag_ptr);
                if (diag != 0.0) {
#pragma unroll
                    for (int i = 0; i < Cfg::NPASS; ++i) {
                        const int r = row_t + rg + i * Cfg::ROWS_PER_PASS;
                        if (r == col) e[i].x += diag;
                        if (r == col + 1) e[i].y += diag;
                    }
                }
            }
            // C tile: the late dependencies of the item hold once the producer has arrived on deps_ok
            mbar_wait(deps_bar(my_slot), my_phase);
            const double* Cp = tk->C;
            if (Cp != nullptr) {
                const double beta = tk->beta;
                const long long ldc = tk->ldc;
                const bool cvec = ((ldc & 1) == 0) && ((reinterpret_cast<uintptr_t>(Cp) & 15) == 0);
                constexpr int CH = (Cfg::NPASS < 8) ? Cfg::NPASS : 8;  // passes fetched at a time (register budget)
#pragma unroll
                for (int i0 = 0; i0 < Cfg::NPASS; i0 += CH) {
                    double2 c[CH];
#pragma unroll
                    for (int ii = 0; ii < CH; ++ii) {
                        const int r = row_t + rg + (i0 + ii) * Cfg::ROWS_PER_PASS;
                        c[ii] = make_double2(0.0, 0.0);
                        if (r < N && col < N) {
                            const double* p = Cp + (long long)r * ldc + col;
                            if (cvec && col + 1 < N) {
                                c[ii] = __ldcg(reinterpret_cast<const double2*>(p));
                            } else {
                                c[ii].x = __ldcg(p);
                                if (col + 1 < N) c[ii].y = __ldcg(p + 1);
                            }
                        }
                    }
#pragma unroll
                    for (int ii = 0; ii < CH; ++ii) {
                        e[i0 + ii].x = fma(beta, c[ii].x, e[i0 + ii].x);
                        e[i0 + ii].y = fma(beta, c[ii].y, e[i0 + ii].y);
                    }
                }
            }
            // accumulators of the item (parked by the consumer warps); product-free items have none
            const bool has_prod = tk->ktiles > 0;
            const double alpha = tk->alpha;
            mbar_wait(accfull_bar, aphase);  // every item goes through the staging hand-shake (the staging tile doubles as
            aphase ^= 1;                     // scratch for the mirror of product-free items)
            double* srow = stg + (size_t)rg * Cfg::STG_LD + 2 * cp;
#pragma unroll
            for (int i = 0; i < Cfg::NPASS; ++i) {
                double2 v = make_double2(0.0, 0.0);
                double* sp = srow + (size_t)(i * Cfg::ROWS_PER_PASS) * Cfg::STG_LD;
                if (has_prod) {
                    v = *reinterpret_cast<const double2*>(sp);
                    if (Cfg::KSPLIT == 2) {
                        const double2 h = *reinterpret_cast<const double2*>(sp + Cfg::STG_HALF);
                        v.x += h.x;
                        v.y += h.y;
                    }
                }
                v.x = fma(alpha, v.x, e[i].x);
                v.y = fma(alpha, v.y, e[i].y);
                const int r = row_t + rg + i * Cfg::ROWS_PER_PASS;
                if (r < N && col < N) {
                    double* p = Out + (long long)r * ldo + col;
                    if (vec && col + 1 < N) {
                        __stcg(reinterpret_cast<double2*>(p), v);
                    } else {
                        __stcg(p, v.x);
                        if (col + 1 < N) __stcg(p + 1, v.y);
                    }
                }
                if (tk->sym) *reinterpret_cast<double2*>(sp) = v;  // finished values, read back by columns below
            }
            if (tk->sym) {
                // Mirror: rows [R0, R0 + 4) x 32 columns of the finished tile go to Out[column][R0 .. R0 + 3] (one 32-byte
                // sector per lane) when the transposed position lies in a tile that is not a work item, i.e. tile
                // (tm', tn') = (C0 / BM, R0 / BN) with tm' BM + BM - 1 < tn' BN (same rule as gemm_dmma.cuh).
                named_bar_sync(2, Cfg::EPI_THREADS);
                const int ew = warp - Cfg::EPI_WARP0;
                constexpr int QUADS = BM / 4, CGROUPS = BN / 32;
                for (int u = ew; u < QUADS * CGROUPS; u += Cfg::EPI_WARPS) {
                    const int q = u / CGROUPS, cg = u - q * CGROUPS;
                    const int R0 = row_t + 4 * q, C0 = col_t + 32 * cg;
                    if (!((C0 / BM) * BM + BM - 1 < (R0 / BN) * BN)) continue;  // warp-uniform
                    const int rr = C0 + lane;                                    // destination row
                    const double* sq = stg + (size_t)(4 * q) * Cfg::STG_LD + 32 * cg + lane;
                    const double a0 = sq[0], a1 = sq[Cfg::STG_LD], a2 = sq[2 * Cfg::STG_LD], a3 = sq[3 * Cfg::STG_LD];
                    if (rr < N && R0 < N) {
                        double* p = Out + (long long)rr * ldo + R0;
                        if (vec && R0 + 3 < N) {
                            __stcg(reinterpret_cast<double2*>(p), make_double2(a0, a1));
                            __stcg(reinterpret_cast<double2*>(p + 2), make_double2(a2, a3));
                        } else {
                            __stcg(p, a0);
                            if (R0 + 1 < N) __stcg(p + 1, a1);
                            if (R0 + 2 < N) __stcg(p + 2, a2);
                            if (R0 + 3 < N) __stcg(p + 3, a3);
                        }
                    }
                }
            }
            // staging tile back to the consumers; completion to the leader, which publishes the item
            __syncwarp();
            if (lane == 0) {
                mbar_arrive(accempty_bar);
                mbar_arrive(epidone_bar(my_slot));
            }
            if (leader) {
                mbar_wait(epidone_bar(my_slot), my_phase);
                fence_acq_rel_gpu();
                publish_tile<BM, BN>(args, ti);
                if (args.trace != nullptr) {
                    TraceRec r;
                    r.task = ti.task; r.tm = ti.tm; r.tn = ti.tn; r.sm = sm_id();
                    r.t_claim = ti.t_claim; r.t_desc = trc[my_slot * 4 + 0]; r.t_first = trc[my_slot * 4 + 1];
                    r.t_kend = trc[my_slot * 4 + 2]; r.t_done = global_ns();
                    args.trace[args.trace_base + ti.item] = r;
                }
                mbar_arrive(tempty_bar(my_slot));
            }
        }
        return;
    }

    if (warp >= Cfg::CONSUMER_WARPS) return;  // warps 9..11 have no role

    // ======================================= consumer warps =======================================
    const int kh = warp / (Cfg::WARPS_M * Cfg::WARPS_N), wq = warp % (Cfg::WARPS_M * Cfg::WARPS_N);
    const int wm = wq / Cfg::WARPS_N, wn = wq % Cfg::WARPS_N;
    const int g = lane >> 2, t = lane & 3;
    uint32_t aoff[2], boff[2];
#pragma unroll
    for (int par = 0; par < 2; ++par) {
        const uint32_t x = par + 2 * t;
        const uint32_t lo = x * 128 + ((((uint32_t)g >> 1) ^ x) << 4) + (g & 1) * 8;
        aoff[par] = (wm * (Cfg::WM / 16)) * SLAB_BYTES + lo;
        boff[par] = Cfg::A_BYTES + (wn * (Cfg::WN / 16)) * SLAB_BYTES + lo;
    }
    // this lane's fragment (i, j) lives at staging row wm WM + 8 i + g, columns wn WN + 8 j + 2 t, + 1
    double* sdst = stg + (size_t)kh * Cfg::STG_HALF + (size_t)(wm * Cfg::WM + g) * Cfg::STG_LD + wn * Cfg::WN + 2 * t;

    int stage = 0;
    uint32_t phase = 0;
    int tslot = 0;
    uint32_t tphase = 0, ephase = 0;
    for (;;) {
        mbar_wait(tfull_bar(tslot), tphase);
        const TileInfo ti = ring[tslot];
        const int ti_slot = tslot;
        const int ti_dep = ti.task ^ ti.tm ^ ti.tn ^ ti.stop ^ ti.item ^ (int)ti.t_claim ^ (int)(ti.t_claim >> 32);
        const int ti_dep_all = (int)__reduce_xor_sync(0xffffffffu, (unsigned)ti_dep);
        if (lane == 0) mbar_arrive_dep(tempty_bar(tslot), ti_dep_all);
        if (++tslot == RING) { tslot = 0; tphase ^= 1; }
        if (ti.stop) break;
        const Task* tk = args.tasks + ti.task;
        const bool tracing = (args.trace != nullptr) && threadIdx.x == 0;
        if (tracing) trc[ti_slot * 4 + 0] = global_ns();
        const int ktiles = tk->ktiles * (tk->ktiles > 0 ? tk->kchunks : 0);
        if (ktiles == 0) {  // product-free item: nothing to park, but the staging hand-shake stays uniform
            if (tracing) { trc[ti_slot * 4 + 1] = global_ns(); trc[ti_slot * 4 + 2] = trc[ti_slot * 4 + 1]; }
            mbar_wait(accempty_bar, ephase ^ 1);
            ephase ^= 1;
            __syncwarp();
            if (lane == 0) mbar_arrive(accfull_bar);
            continue;
        }
        double acc[FM][FN][2];
#pragma unroll
        for (int i = 0; i < FM; ++i)
#pragma unroll
            for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

        // A stage goes back to the producer one iteration late (see gemm_dmma.cuh: the arrive may overtake loads in flight).
        // With two k-halves the halves take ALTERNATE k-tiles of the item (kh = kt & 1), each warp all k4-steps of its
        // stages: the two warps of a scheduler sub-partition (w and w + 4) then work on different stages and one warp's
        // wait behind a stage barrier (barrier, then the LDS latency in front of the first DMMAs: a quarter of the loop's
        // stall samples) is covered by the other's DMMAs.  When both halves shared every stage they reached the barrier
        // together and the DMMA pipe idled for both (per-instruction samples, profiles/r02_ablations.md section 7).
        constexpr bool ALT = (Cfg::KSPLIT == 2);
        constexpr int K4 = BK / 4;
        int prev_stage = -1;
        for (int kt = 0; kt < ktiles; ++kt) {
            if (!ALT || (kt & 1) == kh) {
                mbar_wait(full_bar(stage), phase);
                if (tracing && kt == 0) trc[ti_slot * 4 + 1] = global_ns();
                const uint8_t* sbase = smem + stage * Cfg::STAGE_BYTES;
#pragma unroll
                for (int j = 0; j < K4; ++j) {
                    const int jh = j >> 1, par = j & 1;
                    double a[FM], b[FN];
#pragma unroll
                    for (int i = 0; i < FM; ++i)
                        a[i] = *reinterpret_cast<const double*>(sbase + ((aoff[par] ^ ((i & 1) << 6)) + (i >> 1) * SLAB_BYTES + jh * 1024));
#pragma unroll
                    for (int i = 0; i < FN; ++i)
                        b[i] = *reinterpret_cast<const double*>(sbase + ((boff[par] ^ ((i & 1) << 6)) + (i >> 1) * SLAB_BYTES + jh * 1024));
                    if (j == 0 && prev_stage >= 0) {
                        __syncwarp();
                        if (lane == 0) mbar_arrive(empty_bar(prev_stage));
                    }
#pragma unroll
                    for (int im = 0; im < FM; ++im)
#pragma unroll
                        for (int jn = 0; jn < FN; ++jn) dmma_884(acc[im][jn][0], acc[im][jn][1], a[im], b[jn]);
                }
                prev_stage = stage;
            }
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
        if (prev_stage >= 0) {
            __syncwarp();
            int dep = 0;
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dep ^= __double2hiint(acc[i][j][0]) ^ __double2hiint(acc[i][j][1]);
            if (lane == 0) mbar_arrive_dep(empty_bar(prev_stage), dep);
        }
        if (tracing) trc[ti_slot * 4 + 2] = global_ns();
        // park the accumulators (the epilogue warps have released the staging tile of the previous item long ago)
        mbar_wait(accempty_bar, ephase ^ 1);
        ephase ^= 1;
#pragma unroll
        for (int i = 0; i < FM; ++i)
#pragma unroll
            for (int j = 0; j < FN; ++j)
                *reinterpret_cast<double2*>(sdst + (size_t)(8 * i) * Cfg::STG_LD + 8 * j) = make_double2(acc[i][j][0], acc[i][j][1]);
        __syncwarp();
        if (lane == 0) mbar_arrive(accfull_bar);
    }
}

}  // namespace chebdm
