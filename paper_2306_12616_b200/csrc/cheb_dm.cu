// cheb_dm.cu -- host side of the C ABI declared in include/cheb_dm.h: plan (block sizes, workspace slots,
// TMA descriptors, task/dependency tables) and the launches of the sm_100a kernels.  Product code;
// shares nothing with oracle/.  There is no CPU path: every step of the solve runs in the kernels of
// gemm_dmma.cuh / giant_resident.cuh / aux_kernels.cuh.
#include <cuda.h>
#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>
#include <vector>

#include "../../include/cheb_dm.h"
#include "aux_kernels.cuh"
#include "common.cuh"
#include "gemm_dmma.cuh"
#include "gemm_epi.cuh"
#include "giant_resident.cuh"
#include "ozaki.cuh"

using namespace chebdm;

namespace {

//                 BM   BN  WM  WN  BK  stages  min CTAs/SM
typedef GemmCfg<128, 128, 32, 32, 16, 4, 1> Cfg128x128;   // 16 consumer warps, 128 KB ring, 1 CTA/SM
typedef GemmCfg<128, 64, 32, 32, 16, 4, 2> Cfg128x64;     //  8 consumer warps,  96 KB ring, 2 CTA/SM
typedef GemmCfg<64, 64, 32, 32, 16, 6, 3> Cfg64x64;       //  4 consumer warps,  96 KB ring, 2 CTA/SM (smem)
typedef GemmCfg<64, 32, 16, 16, 32, 8, 1> Cfg64x32w16;    //  8 consumer warps of 16x16, 192 KB ring, 1 CTA/SM
typedef GemmCfg<64, 32, 32, 16, 32, 6, 1> Cfg64x32w32;    //  4 consumer warps of 32x16, 144 KB ring, 1 CTA/SM
typedef GemmCfg<128, 64, 32, 16, 16, 6, 1> Cfg128x64w16;  // 16 consumer warps of 32x16, 144 KB ring, 1 CTA/SM
typedef GemmCfg<32, 32, 16, 16, 32, 6, 2> Cfg32x32;       //  4 consumer warps of 16x16,  96 KB ring, 2 CTA/SM
typedef GemmCfg<64, 64, 32, 16, 32, 6, 1> Cfg64x64w16;    //  8 consumer warps of 32x16, 192 KB ring, 1 CTA/SM
typedef GemmCfg<112, 64, 16, 32, 16, 6, 1> Cfg112x64;     // 14 consumer warps of 16x32, 132 KB ring, 1 CTA/SM (N ~ 1000: 144 tiles)
typedef GemmCfg<64, 32, 16, 16, 32, 4, 2> Cfg64x32x2;     //  8 consumer warps of 16x16,  96 KB ring, 2 CTA/SM (batched small N)
//                BM  BN  WM  WN  k-split BK stages      (gemm_epi.cuh: 8 consumer warps + 4 epilogue warps, 1 CTA/SM)
typedef EpiCfg<64, 32, 32, 16, 2, 32, 7> CfgE64x32;       //  2 k-halves x (2 x 2 warps of 32x16), 168 KB ring + 40 KB staging tile
typedef EpiCfg<64, 64, 32, 16, 1, 32, 5> CfgE64x64;       //  2 x 4 warps of 32x16, 160 KB ring + 36 KB staging tile

enum TileSel { TILE_AUTO = 0, TILE_128x128 = 1, TILE_128x64 = 2, TILE_64x64 = 3, TILE_64x32_W16 = 4, TILE_64x32_W32 = 5,
               TILE_128x64_W16 = 6, TILE_32x32 = 7, TILE_112x64 = 8, TILE_64x64_W16 = 9, TILE_64x32_X2 = 10, TILE_E64x32 = 11, TILE_E64x64 = 12,
               TILE_LAST = 12 };

struct TileShape {
    int BM, BN, BK, box_slabs;
    double eff;  // main-loop efficiency used by the plan-time tile choice (fraction of the DMMA rate, measured)
};
template <class Cfg>
TileShape shape_of(double eff) {
    TileShape t = {Cfg::BM, Cfg::BN, Cfg::BK, Cfg::BOX_SLABS, eff};
    return t;
}
TileShape tile_shape(int sel) {
    switch (sel) {
        case TILE_128x128: return shape_of<Cfg128x128>(0.85);
        case TILE_128x64: return shape_of<Cfg128x64>(0.78);
        case TILE_64x64: return shape_of<Cfg64x64>(0.70);
        case TILE_64x32_W16: return shape_of<Cfg64x32w16>(0.70);
        case TILE_64x32_W32: return shape_of<Cfg64x32w32>(0.65);
        case TILE_32x32: return shape_of<Cfg32x32>(0.60);
        case TILE_64x64_W16: return shape_of<Cfg64x64w16>(0.76);
        case TILE_112x64: return shape_of<Cfg112x64>(0.72);  // 14 consumer warps: two sub-partitions carry 4, two carry 3
        case TILE_64x32_X2: return shape_of<Cfg64x32x2>(0.70);
        case TILE_E64x32: return shape_of<CfgE64x32>(0.88);
        case TILE_E64x64: return shape_of<CfgE64x64>(0.90);
        default: return shape_of<Cfg128x64w16>(0.80);
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (fn) return fn;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess) return nullptr;
    if (qres != cudaDriverEntryPointSuccess) return nullptr;
    fn = reinterpret_cast<EncodeTiledFn>(p);
    return fn;
}

// One grouped launch works on a table: ntl "level tasks" (the products of the method in topological order), each
// instantiated for every slot of the plan: task (lt, slot) at index lt * maxb + slot.  All tasks of a table have the
// same number of work items.
struct TaskTable {
    std::vector<Task> h;
    Task* d;
    int ntl;
    int items_per_task;
    int ctr_task_off, ctr_panel_off;  // this table's regions of the counter block
    int trace_base;
    TaskTable() : d(nullptr), ntl(0), items_per_task(0), ctr_task_off(0), ctr_panel_off(0), trace_base(0) {}
};

}  // namespace

enum { TIMING_SLOTS = 256 };

struct cheb_dm_plan_s {
    int N, M, k, p, Nq, maxb;
    cheb_dm_options_t opt;
    int device, num_sms;
    int tile;  // TileSel actually used
    int BM, BN, BK, box_slabs;
    long long ld;        // padded leading dimension of workspace matrices (multiple of 16)
    long long ldh, ldd;  // leading dimensions of the caller's device matrices
    size_t mat_elems;    // elements per workspace matrix
    int nmat;            // matrices per slot: T_1..T_k | buf0 buf1 buf2 | G_0..G_{p-1} (if any) | U_2..U_{p-1} (if any)
    size_t slot_elems;   // nmat * mat_elems
    int off_G, off_U;    // first matrix of the G / U blocks inside a slot (-1: absent)
    double* ws;          // maxb slots
    // scalar tables (device): costab, Amat, one are shared; the others are per slot
    double *costab, *Amat, *one;
    double *fn, *c, *gT, *dT, *tau, *w;
    double *part;        // front end: per-block (lo, hi)
    double *traces, *gram_part, *gram;  // moments: traces [slot][ntrmat], Gram partials, Gram
    int ntrmat, gram_ctas, gram_passes;
    int front_max_grid;  // co-resident blocks of the cooperative front_end_kernel
    int gemm_per_sm;     // resident CTAs per SM of the product kernel instance of this plan
    int scalar_sums;     // CHEB_DM_SCALAR_SUMS=1 at plan time: FP64-FMA form_sums_kernel (ablation)
    int preformed;       // 1: low-order sums G_l are formed by form_sums_kernel before the giant steps
    int sym;             // 1: symmetric-tile skipping in gemm_dmma_kernel
    short2* sym_tiles;   // device: [sym items] work item -> (tm, tn) of a symmetric task, raster order
    int* sym_panel_target;  // device: [tiles_n] tiles of a symmetric task that write into a column panel (own + mirrored)
    int panel_sym;       // 1: symmetric giant / chain steps wait per column panel (BM a multiple of BN)
    int resident;        // 1: single solves run their giant steps in giant_resident_kernel (small N)
    int moments_on;      // 1: the workspace holds the G and U blocks (cheb_dm_moments / solve / assemble)
    int res_tiles_m, res_tiles_n, res_grid, res_smem;
    DevScalars* sc;      // [maxb]
    CUtensorMap* maps;   // maxb * nmaps_slot descriptors
    int nmaps_slot, map_flatA, map_flatB;
    int tma2d;
    // task tables
    TaskTable baby, giant, chain, flat, misc;
    int* counters;       // device: [error flag | work counters | per-table task_done and panel_done regions]
    size_t counters_ints;
    int nwork, work_next;
    int panel_stride;
    // state
    int have_coeffs, explicit_bounds, have_moments, computed, blocks_nb;
    double beta, mu, a, b;
    int last_launches;
    double flops_per_compute, flops_per_solve;
    size_t ws_bytes;
    // host entry points: two staging sets (H, D, tr D for every slot), copy streams, events
    double *stage_H[2], *stage_D[2], *stage_tr[2];
    cudaStream_t s_in, s_out;
    cudaEvent_t ev_in[2], ev_comp[2], ev_out[2];
    long long n_async;
    int pipe_ready;
    // digit planes of cheb_dm_product_sliced (option sliced = S): [operand][digit][N][oz_kpad] int8, scales [operand][N]
    int oz_S, oz_nsets, oz_solve;   // digit sets: T_1..T_k, the three giant-step buffers (sliced_solve), then the two of the stand-alone product
    long long oz_kpad;
    int8_t* oz_digits;         // [set][digit][N][oz_kpad]
    double* oz_scale;          // [set][N] row scales, then [set][N] diagonal corrections of exact squares
    std::vector<CUtensorMap> oz_maps;  // [set][0: 128-row boxes (left factor), 1: 64-row boxes (right factor)]
    short2* oz_tiles[2];       // raster-ordered tile lists: [0] every tile, [1] the tiles that touch the lower triangle
    int oz_ntiles[2];
    // optional per-tile timeline (cheb_dm_set_trace)
    TraceRec* trace_buf;
    int trace_on, trace_res_base, trace_total, trace_nb;  // trace_nb: matrices of the last traced launch
    // optional timing of the product launches (cheb_dm_set_timing)
    int timing;
    cudaEvent_t ev0[TIMING_SLOTS], ev1[TIMING_SLOTS];  // ring: compute number i uses slot i % TIMING_SLOTS
    long long ev_count;                                // computes recorded since cheb_dm_set_timing(plan, 1)
};

namespace {

#define CUDA_TRY(expr)                                \
    do {                                              \
        cudaError_t e__ = (expr);                     \
        if (e__ != cudaSuccess) return CHEB_DM_ECUDA; \
    } while (0)

// ---- workspace layout: matrix m of slot s ----
double* mat_ptr(const cheb_dm_plan_s* P, int s, int m) { return P->ws + (size_t)s * P->slot_elems + (size_t)m * P->mat_elems; }
double* T_ptr(const cheb_dm_plan_s* P, int s, int n) { return mat_ptr(P, s, n - 1); }             // T_n, 1 <= n <= k
constexpr int NBUF = 3;  // rotating giant-step buffers: B_l lives in buffer l % 3 (see build_tables)
double* buf_ptr(const cheb_dm_plan_s* P, int s, int i) { return mat_ptr(P, s, P->k + i); }        // giant-step buffers
double* G_ptr(const cheb_dm_plan_s* P, int s, int l) { return mat_ptr(P, s, P->off_G + l); }      // G_l, 0 <= l < p
double* U_ptr(const cheb_dm_plan_s* P, int s, int j) {                                            // U_j = T_j(T_k), 1 <= j <= p-1
    return j == 1 ? T_ptr(P, s, P->k) : mat_ptr(P, s, P->off_U + j - 2);
}
int T_map(const cheb_dm_plan_s* P, int s, int n) { return s * P->nmaps_slot + n - 1; }
int buf_map(const cheb_dm_plan_s* P, int s, int i) { return s * P->nmaps_slot + P->k + i; }
int flatA_map(const cheb_dm_plan_s* P, int s, int l) { return s * P->nmaps_slot + P->map_flatA + l - 1; }  // G_l, l >= 1
int flatB_map(const cheb_dm_plan_s* P, int s, int j) { return s * P->nmaps_slot + P->map_flatB + j - 1; }  // U_j, j >= 1

// Algorithm 1, reading A7 for s = 1.  Each entry: T_n = 2 T_l T_r - T_m.
struct BabyProd {
    int n, l, r, m, stage;
};
std::vector<BabyProd> baby_schedule(int k, int pairing) {
    std::vector<BabyProd> v;
    if (k < 2) return v;
    if (pairing == CHEB_DM_PAIR_SERIAL) {
        for (int n = 2; n <= k; ++n) v.push_back({n, 1, n - 1, n - 2, n - 1});
        return v;
    }
    int nstages = 0;
    while ((1 << nstages) < k) ++nstages;
    if (pairing == CHEB_DM_PAIR_BALANCED) {
        // T_n = 2 T_a T_b - T_{a-b}, a = ceil(n/2), b = floor(n/2): same ceil(log2 k) stages and the same concurrency
        // as Algorithm 1 (stage s yields T_{2^{s-1}+1} .. T_{2^s}), the subtracted term is always T_0 or T_1
        for (int s = 1; s <= nstages; ++s)
            for (int n = (1 << (s - 1)) + 1; n <= (1 << s) && n <= k; ++n) v.push_back({n, (n + 1) / 2, n / 2, (n + 1) / 2 - n / 2, s});
        return v;
    }
    for (int s = 1; s <= nstages; ++s) {
        if (s == 1) {
            v.push_back({2, 1, 1, 0, 1});
            continue;
        }
        const int u = 1 << (s - 2), w = 1 << (s - 1);
        for (int i = u + 1; i <= w; ++i)
            if (i + u <= k) v.push_back({i + u, i, u, i - u, s});
        for (int i = u + 1; i <= w; ++i)
            if (i + w <= k) v.push_back({i + w, w, i, w - i, s});
    }
    return v;
}

// cos(pi r / (2 Nq)), r < 4 Nq, from first-octant long-double evaluations (angle reduced exactly).
void build_costab(int Nq, std::vector<double>& tab) {
    tab.resize((size_t)4 * Nq);
    const long double h = 3.14159265358979323846264338327950288L / (2.0L * Nq);
    for (int r = 0; r < 4 * Nq; ++r) {
        int q = r;
        long double sign = 1.0L;
        if (q > 2 * Nq) q = 4 * Nq - q;           // cos(2pi - t) = cos t
        if (q > Nq) { q = 2 * Nq - q; sign = -1.0L; }  // cos(pi - t) = -cos t
        // q in [0, Nq]: angle in [0, pi/2]
        long double v = (2 * q <= Nq) ? cosl(h * q) : sinl(h * (Nq - q));
        if (q == Nq) v = 0.0L;
        tab[r] = (double)(sign * v);
    }
}

// Matrix A of Eq. (10)-(11): T_k^j = sum_l a_{j,l} T_{lk}.  Row-major p x p.
void build_Amat(int p, std::vector<double>& A) {
    A.assign((size_t)p * p, 0.0);
    auto at = [&](int j, int l) -> double& { return A[(size_t)j * p + l]; };
    at(0, 0) = 1.0;
    if (p > 1) at(1, 1) = 1.0;
    for (int j = 2; j < p; ++j) {
        auto prev = [&](int l) { return (l >= 0 && l <= j - 1) ? at(j - 1, l) : 0.0; };
        at(j, 0) = 0.5 * prev(1);
        at(j, 1) = prev(0) + 0.5 * prev(2);
        for (int l = 2; l <= j; ++l) at(j, l) = 0.5 * (prev(l - 1) + prev(l + 1));
    }
}

int ceil_div(int a, int b) { return (a + b - 1) / b; }

// Work items of a product whose result is symmetric: tile (tm, tn) is computed iff it touches the lower triangle,
// tm BM + BM - 1 >= tn BN, i.e. tm >= floor(tn BN / BM); the rest is filled by mirror stores.
int sym_tm0(int tn, int BM, int BN) { return (tn * BN) / BM; }
int sym_items(int N, int BM, int BN) {
    const int tiles_m = ceil_div(N, BM), tiles_n = ceil_div(N, BN);
    int n = 0;
    for (int tn = 0; tn < tiles_n; ++tn) {
        const int tm0 = sym_tm0(tn, BM, BN);
        if (tm0 < tiles_m) n += tiles_m - tm0;
    }
    return n;
}

bool is_epi_tile(int sel) { return sel == TILE_E64x32 || sel == TILE_E64x64; }

void choose_tile(cheb_dm_plan_s* P) {
    int sel = P->opt.tile;
    if (sel < TILE_AUTO || sel > TILE_LAST) sel = TILE_AUTO;
    if (sel == TILE_AUTO) {
        // One product level is the unit of the serial chain (giant steps), so pick the shape that minimises the time of a
        // level on this device: whole waves of work items (all matrices of a batch are claimed together) x tile area /
        // measured main-loop efficiency.  Measured on B200 (profiles/r02_ablations.md):
        //  * the kernel with specialised epilogue warps (gemm_epi.cuh, 64x32 and 64x64 tiles) wins from N ~ 450 up to
        //    N = 5000 (cfg3: 0.90 of the DMMA peak against 0.84 with 128x128 tiles of the generic kernel, whose 18 warps
        //    leave 96 registers per thread): its consumers never wait for an epilogue;
        //  * below that the K loop of an item is shorter than the epilogue warps' work on it: 64x32 tiles of the generic
        //    kernel, or 32x32 tiles with 2 CTAs per SM when a batch level has enough items to fill them;
        //  * single solves at N <= 512 run their giant steps in the resident kernel; the shape only serves the baby steps.
        const bool single_small = (P->maxb == 1 && P->N <= 32 * GR_MAX_KTILES);
        if (single_small) {
            sel = (P->N >= 450) ? TILE_E64x32 : TILE_64x32_W16;
        } else {
            int cand[3], ncand = 0;
            if (P->N >= 450) {
                cand[ncand++] = TILE_E64x32;
                cand[ncand++] = TILE_E64x64;
                if (P->N >= 3000) cand[ncand++] = TILE_128x128;
            } else {
                cand[ncand++] = TILE_64x32_W16;
                if (P->maxb > 1) cand[ncand++] = TILE_32x32;
            }
            // time of one product level in microseconds: whole waves x (K loop of an item at 250 GFLOP/s per SM / measured
            // main-loop efficiency + what is not overlapped per item: 0.3 us with epilogue warps, ~3 us without), plus, when a
            // level is a single wave, the epilogue -> publish -> poll -> TMA tail that no second wave hides
            double best = 0.0;
            for (int c = 0; c < ncand; ++c) {
                const TileShape t = tile_shape(cand[c]);
                const int per_sm = (cand[c] == TILE_32x32) ? 2 : 1;
                const bool epi = is_epi_tile(cand[c]);
                const long long tiles = (long long)(P->sym ? sym_items(P->N, t.BM, t.BN) : ceil_div(P->N, t.BM) * ceil_div(P->N, t.BN)) * P->maxb;
                const long long waves = (tiles + (long long)P->num_sms * per_sm - 1) / ((long long)P->num_sms * per_sm);
                double eff = t.eff;
                if (cand[c] == TILE_E64x32 && P->N > 2500) eff -= 0.03;  // L2 -> SM operand traffic of the narrow tile
                const double kloop = 2.0 * t.BM * t.BN * (double)P->N / 250e3 * per_sm / eff;
                double cost = (double)waves * (kloop + (epi ? 0.3 : 3.0));
                if (waves == 1) cost += epi ? 6.3 : 1.6;
                if (c == 0 || cost < best) {
                    sel = cand[c];
                    best = cost;
                }
            }
        }
    }
    const TileShape t = tile_shape(sel);
    P->tile = sel;
    P->BM = t.BM;
    P->BN = t.BN;
    P->BK = t.BK;
    P->box_slabs = t.box_slabs;
}

Task blank_task(const cheb_dm_plan_s* P, int slot) {
    Task t;
    memset(&t, 0, sizeof(t));
    t.ktiles = ceil_div(P->N, P->BK);
    t.kchunks = 1;
    t.tiles_m = ceil_div(P->N, P->BM);
    t.tiles_n = ceil_div(P->N, P->BN);
    t.nitems = t.tiles_m * t.tiles_n;
    t.slot = slot;
    t.alpha = 1.0;
    t.lds = P->ld;
    t.sum_stride = (long long)P->mat_elems;
    return t;
}

void add_dep(Task& t, int kind, int idx, int target) {
    if (t.ndeps >= MAX_DEPS) return;  // callers never exceed MAX_DEPS
    t.dep_kind[t.ndeps] = kind;
    t.dep_idx[t.ndeps] = idx;
    t.dep_target[t.ndeps] = target;
    ++t.ndeps;
}

void build_tables(cheb_dm_plan_s* P) {
    const int k = P->k, p = P->p, B = P->maxb;
    const int tiles = ceil_div(P->N, P->BM) * ceil_div(P->N, P->BN);
    const int tiles_m = ceil_div(P->N, P->BM);
    // every matrix of the solve is a polynomial of X, hence symmetric: lower-triangle tiles only (option symmetric)
    const int stiles = P->sym ? sym_items(P->N, P->BM, P->BN) : tiles;
    auto idx = [&](int lt, int s) { return lt * B + s; };

    // ---- baby steps: T_n = 2 T_l T_r - T_m (Eq. 7 / 22-23 / Algorithm 1) ----
    const int pairing = (P->opt.pairing == CHEB_DM_PAIR_AUTO) ? CHEB_DM_PAIR_BALANCED : P->opt.pairing;
    std::vector<BabyProd> sched = baby_schedule(k, pairing);
    {
        TaskTable& tt = P->baby;
        tt.ntl = (int)sched.size();
        tt.items_per_task = stiles;
        tt.h.assign((size_t)tt.ntl * B, Task());
        std::vector<int> lt_of(k + 1, -1);  // level task that produces T_n (n >= 2)
        for (int lt = 0; lt < tt.ntl; ++lt) {
            const BabyProd& bp = sched[lt];
            for (int s = 0; s < B; ++s) {
                Task t = blank_task(P, s);
                t.mapA = T_map(P, s, bp.l);
                t.mapB = T_map(P, s, bp.r);
                t.alpha = 2.0;
                if (bp.m == 0) {
                    t.diag_const = -1.0;  // - T_0 = -I
                } else {
                    t.C = T_ptr(P, s, bp.m);
                    t.ldc = P->ld;
                    t.beta = -1.0;
                }
                t.Out = T_ptr(P, s, bp.n);
                t.ldo = P->ld;
                const int deps[3] = {bp.l, bp.r, bp.m};
                for (int d = 0; d < 3; ++d) {
                    const int n = deps[d];
                    if (n < 2) continue;
                    bool dup = false;
                    for (int e = 0; e < d; ++e) dup = dup || (deps[e] == n);
                    if (!dup) add_dep(t, DEP_TASK, idx(lt_of[n], s), stiles);
                }
                t.sym = P->sym;
                t.nitems = stiles;
                tt.h[idx(lt, s)] = t;
            }
            lt_of[bp.n] = lt;
        }
    }

    // ---- giant steps ----
    // CHEBYSHEV: B_l = G_l + 2 Y B_{l+1} - B_{l+2} (l = p-1..1), D = G_0 + Y B_1 - B_2, G_l = sum_i g_{i,l} T_i.
    // POWER    : acc_j = S_j + Y acc_{j+1} (Eq. 4), S_j = sum_i d_{i,j} T_i (Eq. 21).
    // B_l / acc_l lives in buf[l % 3]; Y = T_k.  Without symmetric tiles the column panels of successive steps are
    // independent chains (step l only waits for the SAME column panel of step l+1: DEP_PANEL_N).  With symmetric tiles a
    // column panel also receives the mirror of the row block(s) it crosses, so step l waits until everything step l+1
    // writes into its panel is there (DEP_PANEL_SYM) -- the last wave of a step then overlaps the first of the next, and the
    // publish -> poll -> TMA tail of a step is hidden for all but the last panels.  Three rotating buffers make that safe:
    // step l writes buf[l % 3] (old content B_{l+3}), whose readers are step l+2 (as the streamed operand, any panel: hence
    // the second dependency, on the whole of step l+2, which was claimed two levels earlier and never stalls in practice)
    // and step l+1 (as C, own tile only: the tile of the same panel is complete, and mirror stores only go to tiles that are
    // not work items, which nobody reads as C).  The baby block is complete when this table is launched (stream order).
    {
        const bool power = (P->opt.outer == CHEB_DM_OUTER_POWER);
        TaskTable& tt = P->giant;
        tt.ntl = p;
        const bool gsym = P->sym != 0;
        tt.items_per_task = gsym ? stiles : tiles;
        tt.h.assign((size_t)tt.ntl * B, Task());
        for (int lt = 0; lt < p; ++lt) {
            const int l = p - 1 - lt;
            for (int s = 0; s < B; ++s) {
                const double* coefT = (power ? P->dT : P->gT) + (size_t)s * k * p;
                Task t = blank_task(P, s);
                const bool has_prod = (l + 1 <= p - 1);
                if (has_prod) {
                    t.mapA = T_map(P, s, k);
                    t.mapB = buf_map(P, s, (l + 1) % NBUF);
                    t.alpha = (power || l == 0) ? 1.0 : 2.0;
                    if (!power && l + 2 <= p - 1) {
                        t.C = buf_ptr(P, s, (l + 2) % NBUF);
                        t.ldc = P->ld;
                        t.beta = -1.0;
                    }
                } else {
                    t.ktiles = 0;
                }
                if (l == 0) {
                    t.out_is_user = 1;
                } else {
                    t.Out = buf_ptr(P, s, l % NBUF);
                    t.ldo = P->ld;
                }
                if (P->preformed) {
                    // G_l / S_l was formed beforehand (diagonal term included): one extra tile, weight 1
                    t.sum_base = G_ptr(P, s, l);
                    t.sum_count = 1;
                    t.coef = P->one;
                    t.diag_ptr = nullptr;
                } else {
                    // low-order sum: T_1..T_{k-1} with coefficients row l of the table, T_0 = I through diag_ptr
                    t.sum_base = T_ptr(P, s, 1);
                    t.sum_count = k - 1;
                    t.coef = coefT + (size_t)l * k + 1;
                    t.diag_ptr = coefT + (size_t)l * k;
                }
                t.ndeps_early = 0;
                // (symmetric tiles: a panel also receives mirrored blocks from the tiles of other panels, so the step
                // waits for the whole previous step; the resident kernel has its own counters)
                if (gsym) {
                    t.sym = 1;
                    t.nitems = stiles;
                    if (has_prod) {
                        if (P->panel_sym) {
                            add_dep(t, DEP_PANEL_SYM, idx(lt - 1, s), 0);
                            if (lt >= 2) add_dep(t, DEP_TASK, idx(lt - 2, s), stiles);
                        } else {
                            add_dep(t, DEP_TASK, idx(lt - 1, s), stiles);
                        }
                    }
                } else if (has_prod) {
                    add_dep(t, DEP_PANEL_N, idx(lt - 1, s), tiles_m);
                }
                tt.h[idx(lt, s)] = t;
            }
        }
    }

    // ---- giant block (cheb_dm_moments / cheb_dm_solve): U_j = T_j(Y), U_{j+1} = 2 Y U_j - U_{j-1}, j = 1..p-2, kept in
    // the workspace (U_1 = Y = T_k, U_0 = I).  The baby block is complete when this table is launched. ----
    if (P->moments_on) {
        TaskTable& tt = P->chain;
        tt.ntl = (p >= 3) ? p - 2 : 0;
        tt.items_per_task = stiles;
        tt.h.assign((size_t)tt.ntl * B, Task());
        for (int lt = 0; lt < tt.ntl; ++lt) {
            const int j = lt + 1;
            for (int s = 0; s < B; ++s) {
                Task t = blank_task(P, s);
                t.mapA = T_map(P, s, k);
                t.mapB = flatB_map(P, s, j);
                t.alpha = 2.0;
                if (j == 1) {
                    t.diag_const = -1.0;
                } else {
                    t.C = U_ptr(P, s, j - 1);
                    t.ldc = P->ld;
                    t.beta = -1.0;
                }
                t.Out = U_ptr(P, s, j + 1);
                t.ldo = P->ld;
                t.sym = P->sym;
                t.nitems = stiles;
                // U_{j+1} streams U_j (whole column panel) and reads its own tile of U_{j-1}; every U_j has its own matrix
                if (j >= 2) add_dep(t, (P->sym && P->panel_sym) ? DEP_PANEL_SYM : DEP_TASK, idx(lt - 1, s), stiles);
                tt.h[idx(lt, s)] = t;
            }
        }
        // ---- flat giant step: D = G_0 + sum_{l=1}^{p-1} G_l U_l as ONE long-K product ----
        TaskTable& tf = P->flat;
        tf.ntl = 1;
        tf.items_per_task = stiles;
        tf.h.assign((size_t)B, Task());
        for (int s = 0; s < B; ++s) {
            Task t = blank_task(P, s);
            if (p >= 2) {
                t.mapA = flatA_map(P, s, 1);
                t.mapB = flatB_map(P, s, 1);
                t.kchunks = p - 1;
            } else {
                t.ktiles = 0;
            }
            t.out_is_user = 1;
            t.sum_base = G_ptr(P, s, 0);
            t.sum_count = 1;
            t.coef = P->one;
            t.sym = P->sym;
            t.nitems = stiles;
            tf.h[s] = t;
        }
    }

    // ---- scratch task of cheb_dm_product (slot 0) ----
    {
        TaskTable& tt = P->misc;
        tt.ntl = 1;
        tt.items_per_task = tiles;
        tt.h.assign((size_t)B, Task());
        Task t = blank_task(P, 0);
        t.mapA = buf_map(P, 0, 0);
        t.mapB = buf_map(P, 0, 1);
        t.out_is_user = 1;
        tt.h[0] = t;
    }

    // executed products, counting only the tiles that are computed
    const double res_frac = P->sym ? (double)(P->res_tiles_m + 1) / (2.0 * P->res_tiles_m) : 1.0;  // 32x32 lower-triangle tiles
    const double frac = (double)stiles / (double)tiles;
    const double n3 = 2.0 * (double)P->N * (double)P->N * (double)P->N;
    const double nbaby = (double)P->baby.ntl * frac;
    const double ngiant = (p >= 2) ? (double)(p - 1) * (P->resident ? res_frac : frac) : 0.0;
    P->flops_per_compute = (nbaby + ngiant) * n3;
    const double ngen = (p >= 2) ? (double)(p - 1) * frac : 0.0;
    const double gram_flops = 2.0 * (double)P->N * (double)P->ld * (double)(p > 1 ? p - 1 : 0) * (double)(k > 1 ? k - 1 : 0);
    P->flops_per_solve = (nbaby + (double)P->chain.ntl * frac + ngen) * n3 + gram_flops;
}

cheb_dm_status_t encode_one(EncodeTiledFn enc, const cheb_dm_plan_s* P, CUtensorMap* out, void* base, int want2d) {
    CUresult r;
    if (!want2d) {
        // {16 columns (128 B), N rows, ld/16 slabs}: a box of box_slabs slabs x BK rows lands in shared memory as
        // [slab][row][128 B] with the 128-byte swizzle keyed on the row.
        cuuint64_t dims[3] = {16, (cuuint64_t)P->N, (cuuint64_t)(P->ld / 16)};
        cuuint64_t strides[2] = {(cuuint64_t)P->ld * 8, 128};
        cuuint32_t box[3] = {16, (cuuint32_t)P->BK, (cuuint32_t)P->box_slabs};
        cuuint32_t estr[3] = {1, 1, 1};
        r = enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    } else {
        cuuint64_t dims[2] = {(cuuint64_t)P->ld, (cuuint64_t)P->N};
        cuuint64_t strides[1] = {(cuuint64_t)P->ld * 8};
        cuuint32_t box[2] = {16, (cuuint32_t)P->BK};
        cuuint32_t estr[2] = {1, 1};
        r = enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    }
    return r == CUDA_SUCCESS ? CHEB_DM_OK : CHEB_DM_ECUDA;
}

// Operand descriptors of slot s: T_1..T_k, buf0, buf1, then (moments_on) G_1..G_{p-1} and U_1..U_{p-1} as two
// contiguous runs for the long-K product (U_1's entry describes T_k again).
cheb_dm_status_t encode_maps(cheb_dm_plan_s* P) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return CHEB_DM_ECUDA;
    const int nmaps = P->nmaps_slot * P->maxb;
    std::vector<CUtensorMap> h(nmaps);
    const char* env2d = getenv("CHEB_DM_TMA2D");
    int want2d = (env2d && env2d[0] == '1') ? 1 : 0;
    for (int pass = 0; pass < 2; ++pass) {
        bool ok = true;
        for (int s = 0; s < P->maxb && ok; ++s) {
            CUtensorMap* hs = h.data() + (size_t)s * P->nmaps_slot;
            for (int i = 0; i < P->k + NBUF && ok; ++i) ok = encode_one(enc, P, hs + i, mat_ptr(P, s, i), want2d) == CHEB_DM_OK;
            if (P->moments_on)
                for (int l = 1; l <= P->p - 1 && ok; ++l) {
                    ok = encode_one(enc, P, hs + P->map_flatA + l - 1, G_ptr(P, s, l), want2d) == CHEB_DM_OK &&
                         encode_one(enc, P, hs + P->map_flatB + l - 1, U_ptr(P, s, l), want2d) == CHEB_DM_OK;
                }
        }
        if (ok) {
            P->tma2d = want2d;
            CUDA_TRY(cudaMemcpy(P->maps, h.data(), sizeof(CUtensorMap) * nmaps, cudaMemcpyHostToDevice));
            return CHEB_DM_OK;
        }
        if (want2d) break;
        want2d = 1;  // the driver refused the slab view: fall back to one 2-D box per slab
    }
    return CHEB_DM_ECUDA;
}

// Per plan (and therefore per device): opt in to the dynamic shared memory of the product kernel instance and record
// how many of its CTAs fit an SM.
template <class Cfg>
cheb_dm_status_t prepare_inst(int* per_sm) {
    CUDA_TRY(cudaFuncSetAttribute(gemm_dmma_kernel<Cfg>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, gemm_dmma_kernel<Cfg>, Cfg::THREADS, Cfg::SMEM_BYTES));
    return *per_sm >= 1 ? CHEB_DM_OK : CHEB_DM_ECUDA;
}
template <class Cfg>
cheb_dm_status_t prepare_epi(int* per_sm) {
    CUDA_TRY(cudaFuncSetAttribute(gemm_epi_kernel<Cfg>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, gemm_epi_kernel<Cfg>, Cfg::THREADS, Cfg::SMEM_BYTES));
    return *per_sm >= 1 ? CHEB_DM_OK : CHEB_DM_ECUDA;
}
cheb_dm_status_t prepare_gemm(cheb_dm_plan_s* P) {
    switch (P->tile) {
        case TILE_E64x32: return prepare_epi<CfgE64x32>(&P->gemm_per_sm);
        case TILE_E64x64: return prepare_epi<CfgE64x64>(&P->gemm_per_sm);
        case TILE_128x128: return prepare_inst<Cfg128x128>(&P->gemm_per_sm);
        case TILE_128x64: return prepare_inst<Cfg128x64>(&P->gemm_per_sm);
        case TILE_64x64: return prepare_inst<Cfg64x64>(&P->gemm_per_sm);
        case TILE_64x32_W16: return prepare_inst<Cfg64x32w16>(&P->gemm_per_sm);
        case TILE_64x32_W32: return prepare_inst<Cfg64x32w32>(&P->gemm_per_sm);
        case TILE_32x32: return prepare_inst<Cfg32x32>(&P->gemm_per_sm);
        case TILE_112x64: return prepare_inst<Cfg112x64>(&P->gemm_per_sm);
        case TILE_64x64_W16: return prepare_inst<Cfg64x64w16>(&P->gemm_per_sm);
        case TILE_64x32_X2: return prepare_inst<Cfg64x32x2>(&P->gemm_per_sm);
        default: return prepare_inst<Cfg128x64w16>(&P->gemm_per_sm);
    }
}

template <class Cfg>
cheb_dm_status_t launch_inst(const LaunchArgs& la, int grid, cudaStream_t st) {
    gemm_dmma_kernel<Cfg><<<grid, Cfg::THREADS, Cfg::SMEM_BYTES, st>>>(la);
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

template <class Cfg>
cheb_dm_status_t launch_epi(const LaunchArgs& la, int grid, cudaStream_t st) {
    gemm_epi_kernel<Cfg><<<grid, Cfg::THREADS, Cfg::SMEM_BYTES, st>>>(la);
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

// Launch the level tasks [lt0, lt1) of a table for the slots [0, nb) as one persistent grid.
cheb_dm_status_t launch_tasks(cheb_dm_plan_s* P, const TaskTable& tt, int lt0, int lt1, int nb, int use_deps,
                              double* const* userD, long long ldD, cudaStream_t st) {
    if (lt1 <= lt0 || nb < 1) return CHEB_DM_OK;
    LaunchArgs la;
    memset(&la, 0, sizeof(la));
    la.tasks = tt.d;
    la.maps = P->maps;
    la.work_counter = P->counters + 1 + (P->work_next++ % P->nwork);
    la.task_done = P->counters + tt.ctr_task_off;
    la.panel_done = P->counters + tt.ctr_panel_off;
    la.panel_stride = P->panel_stride;
    la.lt_begin = lt0;
    la.lt_end = lt1;
    la.nb = nb;
    la.maxb = P->maxb;
    la.items_per_task = tt.items_per_task;
    la.use_deps = use_deps;
    la.N = P->N;
    for (int s = 0; s < nb; ++s) la.userD[s] = userD ? userD[s] : nullptr;
    la.ldD = ldD;
    la.tma2d = P->tma2d;
    la.sym_tiles = P->sym_tiles;
    la.sym_panel_target = P->sym_panel_target;
    la.error_flag = P->counters;
    la.trace = P->trace_on ? P->trace_buf : nullptr;
    la.trace_base = tt.trace_base + lt0 * tt.items_per_task * nb;  // a table's region holds ntl * maxb * items records
    if (P->trace_on) P->trace_nb = nb;
    const long long items = (long long)(lt1 - lt0) * nb * tt.items_per_task;
    long long grid = (long long)P->gemm_per_sm * P->num_sms;
    if (grid > items) grid = items;
    if (grid < 1) grid = 1;
    ++P->last_launches;
    switch (P->tile) {
        case TILE_E64x32: return launch_epi<CfgE64x32>(la, (int)grid, st);
        case TILE_E64x64: return launch_epi<CfgE64x64>(la, (int)grid, st);
        case TILE_128x128: return launch_inst<Cfg128x128>(la, (int)grid, st);
        case TILE_128x64: return launch_inst<Cfg128x64>(la, (int)grid, st);
        case TILE_64x64: return launch_inst<Cfg64x64>(la, (int)grid, st);
        case TILE_64x32_W16: return launch_inst<Cfg64x32w16>(la, (int)grid, st);
        case TILE_64x32_W32: return launch_inst<Cfg64x32w32>(la, (int)grid, st);
        case TILE_32x32: return launch_inst<Cfg32x32>(la, (int)grid, st);
        case TILE_112x64: return launch_inst<Cfg112x64>(la, (int)grid, st);
        case TILE_64x64_W16: return launch_inst<Cfg64x64w16>(la, (int)grid, st);
        case TILE_64x32_X2: return launch_inst<Cfg64x32x2>(la, (int)grid, st);
        default: return launch_inst<Cfg128x64w16>(la, (int)grid, st);
    }
}

// A whole table: one persistent launch (GROUPED), or one launch per level task (SERIAL: the paper's single-stream
// mode, PAPER.md:190 -- the ablation baseline).
cheb_dm_status_t run_table(cheb_dm_plan_s* P, const TaskTable& tt, int nb, double* const* userD, long long ldD, cudaStream_t st) {
    if (tt.ntl <= 0) return CHEB_DM_OK;
    if (P->opt.sched == CHEB_DM_SCHED_GROUPED) return launch_tasks(P, tt, 0, tt.ntl, nb, 1, userD, ldD, st);
    for (int lt = 0; lt < tt.ntl; ++lt) {
        cheb_dm_status_t s = launch_tasks(P, tt, lt, lt + 1, nb, 0, userD, ldD, st);
        if (s != CHEB_DM_OK) return s;
    }
    return CHEB_DM_OK;
}

bool device_ok(const cheb_dm_plan_s* P) {
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev == P->device;
}

int front_grid_for(const cheb_dm_plan_s* P, int nb) {
    int want = ceil_div(P->N, 16);
    const int kp = P->k * P->p;
    if (ceil_div(kp, 16) > want) want = ceil_div(kp, 16);
    if (ceil_div(P->Nq, 512) > want) want = ceil_div(P->Nq, 512);
    long long g = (long long)want * nb;
    if (g > P->front_max_grid) g = P->front_max_grid;
    if (g < nb) g = nb;
    return (int)g;
}

// Steps a-1 .. a-3 on the stream, one cooperative launch over the nb matrices: counters reset, bounds (+ rescale of H
// into T_1), c_n, g (and d).  do_bounds / do_coeffs select the halves (cheb_dm_solve runs them apart).
cheb_dm_status_t front_end(cheb_dm_plan_s* P, int nb, const double* const* dH, long long ldh, const double* mu, int do_bounds,
                           int do_coeffs, int mu_from_device, cudaStream_t st) {
    FrontArgs fa;
    memset(&fa, 0, sizeof(fa));
    fa.nb = nb;
    fa.N = P->N;
    for (int s = 0; s < nb; ++s) {
        fa.H[s] = dH ? dH[s] : nullptr;
        fa.mu[s] = mu ? mu[s] : P->mu;
    }
    fa.ldh = ldh;
    fa.X = T_ptr(P, 0, 1);
    fa.slot_stride = (long long)P->slot_elems;
    fa.ldx = P->ld;
    fa.sc = P->sc;
    fa.explicit_bounds = P->explicit_bounds;
    fa.a = P->a;
    fa.b = P->b;
    fa.part = P->part;
    fa.counters = P->counters + 1;  // [0] is the sticky error flag
    fa.ncounters = (int)P->counters_ints - 1;
    {
        // rows are dealt to the blocks of a matrix in rounds of 16 / segs rows; segs = the power of two that minimises
        // rounds x elements per warp and round
        const int grid = front_grid_for(P, nb);
        const int sblocks = grid / nb > 0 ? grid / nb : 1;
        long long best = -1;
        fa.segs = 1;
        for (int sg = 1; sg <= 16; sg *= 2) {
            const long long rounds = ceil_div(P->N, sblocks * (16 / sg));
            const long long cost = rounds * ceil_div(P->N, sg);
            if (best < 0 || cost < best) { best = cost; fa.segs = sg; }
        }
    }
    fa.do_bounds = do_bounds;
    fa.do_coeffs = do_coeffs;
    fa.mu_from_device = mu_from_device;
    fa.beta = P->beta;
    fa.costab = P->costab;
    fa.Nq = P->Nq;
    fa.M = P->M;
    fa.fn = P->fn;
    fa.c = P->c;
    fa.k = P->k;
    fa.p = P->p;
    fa.Amat = P->Amat;
    fa.want_d = (P->opt.outer == CHEB_DM_OUTER_POWER) ? 1 : 0;
    fa.gT = P->gT;
    fa.dT = P->dT;
    void* args[] = {(void*)&fa};
    CUDA_TRY(cudaLaunchCooperativeKernel((const void*)front_end_kernel, dim3(front_grid_for(P, nb)), dim3(512), args, 0, st));
    P->work_next = 0;
    ++P->last_launches;
    return CHEB_DM_OK;
}

// Low-order sums G_l = sum_i coef_{i,l} T_i of Eq. (21) for all l at once (a-5, batched form), nb matrices.
// full = true: every element (the G_l are operands of the long-K product); false: only the tiles the giant steps read.
// cheb_tables: the sums multiply U_l = T_l(T_k) (long-K assembly of cheb_dm_solve / cheb_dm_assemble), so their coefficients
// are the Chebyshev table g whatever the outer recursion of the plan.
cheb_dm_status_t form_sums(cheb_dm_plan_s* P, int nb, bool full, int tileM, int tileN, cudaStream_t st, bool cheb_tables = false) {
    const double* coefT = (P->opt.outer == CHEB_DM_OUTER_POWER && !cheb_tables) ? P->dT : P->gT;
    const int symBM = (P->sym && !full) ? tileM : 0;
    if (P->scalar_sums) {  // FP64-FMA version (ablation)
        const long long pairs = (long long)P->N * P->ld / 2;
        dim3 grid((unsigned)((pairs + 255) / 256), (unsigned)ceil_div(P->p, SUMS_CHUNK), (unsigned)nb);
        form_sums_kernel<<<grid, 256, sizeof(double) * P->k * SUMS_CHUNK, st>>>(T_ptr(P, 0, 1), (long long)P->mat_elems, P->ld, P->N, P->k, P->p,
                                                                              coefT, G_ptr(P, 0, 0), symBM, tileN, (long long)P->slot_elems);
    } else {
        const long long warps = ((long long)P->N * P->ld + 31) / 32;
        dim3 grid((unsigned)((warps + 7) / 8), (unsigned)ceil_div(P->p, SUMS_CHUNK), (unsigned)nb);
        const size_t smem = sizeof(double) * (size_t)((((P->k - 1) + 3) & ~3) + 1) * SUMS_CHUNK;
        form_sums_dmma_kernel<<<grid, 256, smem, st>>>(T_ptr(P, 0, 1), (long long)P->mat_elems, P->ld, P->N, P->k, P->p, coefT, G_ptr(P, 0, 0),
                                                       symBM, tileN, (long long)P->slot_elems);
    }
    ++P->last_launches;
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

// Giant steps of ONE solve in the resident-multiplier kernel (slot 0 of the giant table); cooperative launch because
// its CTAs wait on one another's panel counters.
cheb_dm_status_t run_giant_resident(cheb_dm_plan_s* P, double* userD, long long ldD, cudaStream_t st) {
    GiantArgs ga;
    memset(&ga, 0, sizeof(ga));
    ga.tasks = P->giant.d;
    ga.maps = P->maps;
    ga.first_task = 0;
    ga.nsteps = P->giant.ntl;
    ga.task_stride = P->maxb;
    ga.N = P->N;
    ga.ktiles = ceil_div(P->N, GR_BK);
    ga.tiles_m = P->res_tiles_m;
    ga.tiles_n = P->res_tiles_n;
    ga.panel_done = P->counters + P->giant.ctr_panel_off;
    ga.panel_stride = P->panel_stride;
    ga.userD = userD;
    ga.ldD = ldD;
    ga.tma2d = P->tma2d;
    ga.error_flag = P->counters;
    ga.trace = P->trace_on ? P->trace_buf : nullptr;
    ga.trace_base = P->trace_res_base;
    ga.coefT = (P->opt.outer == CHEB_DM_OUTER_POWER) ? P->dT : P->gT;
    ga.Tbase = T_ptr(P, 0, 1);
    ga.Gbase = G_ptr(P, 0, 0);
    ga.mat_stride = (long long)P->mat_elems;
    ga.ld = P->ld;
    ga.k = P->k;
    ga.sym = P->sym;
    void* args[] = {(void*)&ga};
    CUDA_TRY(cudaLaunchCooperativeKernel((const void*)giant_resident_kernel, dim3(P->res_grid), dim3(GR_THREADS), args,
                                         (size_t)P->res_smem, st));
    ++P->last_launches;
    return CHEB_DM_OK;
}

// Products of a fixed-mu solve after the front end: baby steps, sums, giant steps.
cheb_dm_status_t run_products_sliced(cheb_dm_plan_s* P, double* userD, long long ldd, cudaStream_t st);

cheb_dm_status_t run_products(cheb_dm_plan_s* P, int nb, double* const* dD, long long ldd, cudaStream_t st) {
    if (P->oz_solve) return run_products_sliced(P, dD[0], ldd, st);
    cheb_dm_status_t s = run_table(P, P->baby, nb, dD, ldd, st);
    if (s != CHEB_DM_OK) return s;
    if (P->resident && nb == 1) return run_giant_resident(P, dD[0], ldd, st);
    if (P->preformed) {
        s = form_sums(P, nb, false, P->BM, P->BN, st);
        if (s != CHEB_DM_OK) return s;
    }
    return run_table(P, P->giant, nb, dD, ldd, st);
}

cheb_dm_status_t compute_impl(cheb_dm_plan_s* P, int nb, const double* const* dH, long long ldh, double* const* dD, long long ldd,
                              const double* mu, cudaStream_t st) {
    P->last_launches = 0;
    cheb_dm_status_t s = front_end(P, nb, dH, ldh, mu, 1, 1, 0, st);  // also zeroes the scheduler counters
    if (s != CHEB_DM_OK) return s;
    const int slot = (int)(P->ev_count % TIMING_SLOTS);
    if (P->timing) CUDA_TRY(cudaEventRecord(P->ev0[slot], st));
    s = run_products(P, nb, dD, ldd, st);
    if (s != CHEB_DM_OK) return s;
    if (P->timing) {
        CUDA_TRY(cudaEventRecord(P->ev1[slot], st));
        ++P->ev_count;
    }
    P->computed = 1;
    P->blocks_nb = 0;  // the baby block in the workspace no longer belongs to a moments / solve call
    P->have_moments = 0;
    return CHEB_DM_OK;
}

// Baby block, giant block and moments of nb matrices (front end with bounds already run).
cheb_dm_status_t sliced_baby(cheb_dm_plan_s* P, cudaStream_t st);
cheb_dm_status_t sliced_giant(cheb_dm_plan_s* P, double* userD, long long ldd, cudaStream_t st);
cheb_dm_status_t sliced_table(cheb_dm_plan_s* P, const TaskTable& tt, int kind, double* userD, long long ldd, cudaStream_t st);

cheb_dm_status_t blocks_and_moments(cheb_dm_plan_s* P, int nb, cudaStream_t st) {
    cheb_dm_status_t s;
    if (P->oz_solve) {  // the blocks on the sliced int8 path (their FP64 results feed the Gram kernel as usual)
        s = sliced_baby(P, st);
        if (s != CHEB_DM_OK) return s;
        s = sliced_table(P, P->chain, 2 /* SLICED_CHAIN */, nullptr, 0, st);
    } else {
        s = run_table(P, P->baby, nb, nullptr, 0, st);
        if (s != CHEB_DM_OK) return s;
        s = run_table(P, P->chain, nb, nullptr, 0, st);
    }
    if (s != CHEB_DM_OK) return s;
    const int k = P->k, p = P->p;
    diag_traces_kernel<<<dim3(P->ntrmat, nb), 256, 0, st>>>(T_ptr(P, 0, 1), P->off_U >= 0 ? mat_ptr(P, 0, P->off_U) : T_ptr(P, 0, 1),
                                                           (long long)P->mat_elems, (long long)P->slot_elems, P->ld, P->N, k, P->traces, P->ntrmat);
    ++P->last_launches;
    if (p >= 2 && k >= 2) {
        const double* Tb = T_ptr(P, 0, 1);
        const double* Ub = P->off_U >= 0 ? mat_ptr(P, 0, P->off_U) : T_ptr(P, 0, 1);
        const dim3 ggrid(P->gram_ctas, P->gram_passes, nb);
        const int side = (p - 1 > k - 1) ? p - 1 : k - 1;
        if (side <= 8)
            gram_kernel<1><<<ggrid, 256, 0, st>>>(Tb, Ub, (long long)P->mat_elems, (long long)P->slot_elems, (long long)P->N * P->ld, k, p, P->gram_part);
        else if (side <= 16)
            gram_kernel<2><<<ggrid, 256, 0, st>>>(Tb, Ub, (long long)P->mat_elems, (long long)P->slot_elems, (long long)P->N * P->ld, k, p, P->gram_part);
        else
            gram_kernel<4><<<ggrid, 256, 0, st>>>(Tb, Ub, (long long)P->mat_elems, (long long)P->slot_elems, (long long)P->N * P->ld, k, p, P->gram_part);
        ++P->last_launches;
    }
    moments_kernel<<<nb, 1024, 0, st>>>(P->traces, P->ntrmat, P->gram_part, P->gram_ctas, P->gram_passes, P->gram, k, p, P->N, P->tau);
    ++P->last_launches;
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

cheb_dm_status_t bisect(cheb_dm_plan_s* P, int nb, double beta, const double* n_occ, int iters, cudaStream_t st) {
    BisectArgs ba;
    memset(&ba, 0, sizeof(ba));
    for (int s = 0; s < nb; ++s) ba.n_occ[s] = n_occ[s];
    mu_weights_kernel<<<dim3(P->Nq, nb), 128, 0, st>>>(P->tau, P->costab, P->Nq, P->M, P->k * P->p, P->w);
    mu_bisect_kernel<<<nb, 512, 0, st>>>(P->sc, beta, ba, iters, P->costab, P->Nq, P->w);
    P->last_launches += 2;
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

// D from the blocks in the workspace: coefficient tables (mu given, or the device's), sums, one long-K product.
cheb_dm_status_t assemble_impl(cheb_dm_plan_s* P, int nb, const double* mu, int mu_from_device, double* const* dD, long long ldd,
                               cudaStream_t st) {
    cheb_dm_status_t s = front_end(P, nb, nullptr, 0, mu, 0, 1, mu_from_device, st);
    if (s != CHEB_DM_OK) return s;
    // sliced path: the nested giant steps on the digit sets left by the blocks (T_k; the accumulators are re-sliced)
    if (P->oz_solve) return sliced_giant(P, dD[0], ldd, st);
    s = form_sums(P, nb, true, P->BM, P->BN, st, true);
    if (s != CHEB_DM_OK) return s;
    return run_table(P, P->flat, nb, dD, ldd, st);
}

cheb_dm_status_t trace_impl(cheb_dm_plan_s* P, int nb, const double* const* dD, long long ldd, double* out, cudaStream_t st) {
    TraceArgs ta;
    memset(&ta, 0, sizeof(ta));
    for (int s = 0; s < nb; ++s) ta.D[s] = dD[s];
    trace_kernel<<<nb, 1024, 0, st>>>(ta, P->N, ldd, out);
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

// Staging sets of the host entry points: `sets` of them (1 or 2); 2 also creates the copy streams and events.
cheb_dm_status_t ensure_staging(cheb_dm_plan_s* P, int sets) {
    const size_t bytes = sizeof(double) * (size_t)P->N * P->N * P->maxb;
    for (int i = 0; i < sets; ++i) {
        if (P->stage_H[i]) continue;
        const bool ok = cudaMalloc(&P->stage_H[i], bytes) == cudaSuccess && cudaMalloc(&P->stage_D[i], bytes) == cudaSuccess &&
                        cudaMalloc(&P->stage_tr[i], sizeof(double) * P->maxb) == cudaSuccess;
        if (!ok) { cudaGetLastError(); return CHEB_DM_EALLOC; }
        P->ws_bytes += 2 * bytes;
    }
    if (sets >= 2 && !P->pipe_ready) {
        CUDA_TRY(cudaStreamCreateWithFlags(&P->s_in, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamCreateWithFlags(&P->s_out, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CUDA_TRY(cudaEventCreateWithFlags(&P->ev_in[i], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&P->ev_comp[i], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&P->ev_out[i], cudaEventDisableTiming));
        }
        P->pipe_ready = 1;
    }
    return CHEB_DM_OK;
}

bool batch_args_ok(const cheb_dm_plan_s* P, int nb, const double* const* A, double* const* B, const double* mu) {
    if (nb < 1 || nb > P->maxb || !A || !B) return false;
    for (int s = 0; s < nb; ++s) {
        if (!A[s] || !B[s] || A[s] == B[s]) return false;
        if (mu && !isfinite(mu[s])) return false;
        for (int t = 0; t < s; ++t)
            if (B[t] == B[s]) return false;
    }
    return true;
}

// Digit planes, scales and TMA descriptors of cheb_dm_product_sliced.
cheb_dm_status_t prepare_sliced(cheb_dm_plan_s* P) {
    const size_t plane = (size_t)P->N * (size_t)P->oz_kpad;
    P->oz_nsets = (P->oz_solve ? P->k + NBUF + ((P->moments_on && P->p >= 3) ? P->p - 2 : 0) : 0) + 2;
    const size_t bytes = (size_t)P->oz_nsets * (size_t)P->oz_S * plane;
    if (cudaMalloc(&P->oz_digits, bytes) != cudaSuccess || cudaMalloc(&P->oz_scale, sizeof(double) * 2 * P->oz_nsets * P->N) != cudaSuccess) {
        cudaGetLastError();
        return CHEB_DM_EALLOC;
    }
    P->ws_bytes += bytes + sizeof(double) * 2 * P->oz_nsets * P->N;
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return CHEB_DM_ECUDA;
    P->oz_maps.resize((size_t)P->oz_nsets * 2);
    for (int set = 0; set < P->oz_nsets; ++set)
        for (int role = 0; role < 2; ++role) {
            // {k (bytes), row, digit}: a box is one k-block of 64 int8 x 128 (or 64) rows of one digit plane, 64-byte swizzle
            cuuint64_t dims[3] = {(cuuint64_t)P->oz_kpad, (cuuint64_t)P->N, (cuuint64_t)P->oz_S};
            cuuint64_t strides[2] = {(cuuint64_t)P->oz_kpad, (cuuint64_t)plane};
            cuuint32_t box[3] = {(cuuint32_t)OZ_BK, (cuuint32_t)(role == 0 ? OZ_BM : OZ_BN), 1};
            cuuint32_t estr[3] = {1, 1, 1};
            CUresult r = enc(&P->oz_maps[(size_t)set * 2 + role], CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, P->oz_digits + (size_t)set * P->oz_S * plane, dims,
                             strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) return CHEB_DM_ECUDA;
        }
    {
        const int tiles_m = ceil_div(P->N, OZ_BM), tiles_n = ceil_div(P->N, OZ_BN);
        for (int sym = 0; sym < 2; ++sym) {
            std::vector<short2> list;
            for (int band = 0; band * OZ_BAND < tiles_n; ++band)
                for (int tm = 0; tm < tiles_m; ++tm)
                    for (int tn = band * OZ_BAND; tn < tiles_n && tn < (band + 1) * OZ_BAND; ++tn)
                        if (!sym || tm * OZ_BM + OZ_BM - 1 >= tn * OZ_BN) list.push_back(make_short2((short)tm, (short)tn));
            P->oz_ntiles[sym] = (int)list.size();
            if (cudaMalloc(&P->oz_tiles[sym], sizeof(short2) * list.size()) != cudaSuccess) { cudaGetLastError(); return CHEB_DM_EALLOC; }
            CUDA_TRY(cudaMemcpy(P->oz_tiles[sym], list.data(), sizeof(short2) * list.size(), cudaMemcpyHostToDevice));
        }
    }
    switch (P->oz_S) {
        case 2: CUDA_TRY(cudaFuncSetAttribute(oz_gemm_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz_smem_bytes())); break;
        case 3: CUDA_TRY(cudaFuncSetAttribute(oz_gemm_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz_smem_bytes())); break;
        case 4: CUDA_TRY(cudaFuncSetAttribute(oz_gemm_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz_smem_bytes())); break;
        case 5: CUDA_TRY(cudaFuncSetAttribute(oz_gemm_kernel<5>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz_smem_bytes())); break;
        case 6: CUDA_TRY(cudaFuncSetAttribute(oz_gemm_kernel<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz_smem_bytes())); break;
        case 7: CUDA_TRY(cudaFuncSetAttribute(oz_gemm_kernel<7>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz_smem_bytes())); break;
        default: CUDA_TRY(cudaFuncSetAttribute(oz_gemm_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, oz_smem_bytes())); break;
    }
    return CHEB_DM_OK;
}

// Digits of an FP64 matrix (leading dimension ld) into digit set `set`.
cheb_dm_status_t oz_split(cheb_dm_plan_s* P, int set, const double* src, long long ld, cudaStream_t st) {
    const size_t plane = (size_t)P->N * (size_t)P->oz_kpad;
    {
        int8_t* dig = P->oz_digits + (size_t)set * P->oz_S * plane;
        double* sc = P->oz_scale + (size_t)set * P->N;
        double* cr = P->oz_scale + (size_t)(P->oz_nsets + set) * P->N;
        const int passes = (int)((P->oz_kpad + 1023) / 1024);
#define OZ_SPLIT_REG(PS) oz_split_reg_kernel<PS><<<P->N, 256, 0, st>>>(src, ld, P->N, P->oz_S, dig, P->oz_kpad, sc, cr)
        switch (passes) {  // rows up to 6144 elements stay in registers between the maximum and the digits
            case 1: OZ_SPLIT_REG(1); break;
            case 2: OZ_SPLIT_REG(2); break;
            case 3: OZ_SPLIT_REG(3); break;
            case 4: OZ_SPLIT_REG(4); break;
            case 5: OZ_SPLIT_REG(5); break;
            case 6: OZ_SPLIT_REG(6); break;
            default: oz_split_kernel<<<P->N, 256, 0, st>>>(src, ld, P->N, P->oz_S, dig, P->oz_kpad, sc, cr);
        }
#undef OZ_SPLIT_REG
    }
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

// Out = alpha A B + beta C + G + diag I from the digit sets of A and B (oa carries the epilogue operands).
cheb_dm_status_t oz_gemm(cheb_dm_plan_s* P, int setA, int setB, OzArgs oa, int symmetric, cudaStream_t st) {
    const int S = P->oz_S;
    oa.N = P->N;
    oa.S = S;
    oa.kblocks = (int)(P->oz_kpad / OZ_BK);
    oa.tiles_m = ceil_div(P->N, OZ_BM);
    oa.tiles_n = ceil_div(P->N, OZ_BN);
    oa.scaleA = P->oz_scale + (size_t)setA * P->N;
    oa.scaleB = P->oz_scale + (size_t)setB * P->N;
    oa.corr = (setA == setB) ? P->oz_scale + (size_t)(P->oz_nsets + setA) * P->N : nullptr;
    oa.sym = symmetric ? 1 : 0;
    oa.ntiles = P->oz_ntiles[oa.sym];
    oa.tile_list = P->oz_tiles[oa.sym];
    int grid = oa.ntiles;
    if (grid > P->num_sms) grid = P->num_sms;
    const CUtensorMap& mA = P->oz_maps[(size_t)setA * 2];
    const CUtensorMap& mB = P->oz_maps[(size_t)setB * 2 + 1];
    switch (S) {
        case 2: oz_gemm_kernel<2><<<grid, OZ_THREADS, oz_smem_bytes(), st>>>(mA, mB, oa); break;
        case 3: oz_gemm_kernel<3><<<grid, OZ_THREADS, oz_smem_bytes(), st>>>(mA, mB, oa); break;
        case 4: oz_gemm_kernel<4><<<grid, OZ_THREADS, oz_smem_bytes(), st>>>(mA, mB, oa); break;
        case 5: oz_gemm_kernel<5><<<grid, OZ_THREADS, oz_smem_bytes(), st>>>(mA, mB, oa); break;
        case 6: oz_gemm_kernel<6><<<grid, OZ_THREADS, oz_smem_bytes(), st>>>(mA, mB, oa); break;
        case 7: oz_gemm_kernel<7><<<grid, OZ_THREADS, oz_smem_bytes(), st>>>(mA, mB, oa); break;
        default: oz_gemm_kernel<8><<<grid, OZ_THREADS, oz_smem_bytes(), st>>>(mA, mB, oa); break;
    }
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

// Digit set of a workspace matrix of slot 0: T_1..T_k and the three giant-step buffers keep their matrix index, the giant
// block U_2..U_{p-1} follows.
int oz_set_of_matrix(const cheb_dm_plan_s* P, int m) {
    if (m < P->k + NBUF) return m;
    return P->k + NBUF + (m - P->off_U);
}
// ... and of an operand given by its tensor-map index (T_1..T_k, buffers, then the U_1..U_{p-1} run of the long-K product).
int oz_set_of_map(const cheb_dm_plan_s* P, int idx) {
    if (idx < P->k + NBUF) return idx;
    const int j = idx - P->map_flatB + 1;  // U_j; U_1 = T_k
    return j == 1 ? P->k - 1 : P->k + NBUF + (j - 2);
}

enum SlicedKind { SLICED_BABY = 0, SLICED_GIANT = 1, SLICED_CHAIN = 2 };

// One task table on the sliced int8 path (option sliced_solve): the same tasks as the DMMA path (Algorithm 1 / balanced
// pairing for the baby steps, Eq. 4 or its Clenshaw form for the giant steps, U_{j+1} = 2 Y U_j - U_{j-1} for the giant
// block), one launch per product; every result that is an operand later on is sliced once, right after it is formed.
cheb_dm_status_t sliced_table(cheb_dm_plan_s* P, const TaskTable& tt, int kind, double* userD, long long ldd, cudaStream_t st) {
    const int k = P->k;
    cheb_dm_status_t s = CHEB_DM_OK;
    for (int lt = 0; lt < tt.ntl; ++lt) {
        const Task& t = tt.h[(size_t)lt * P->maxb];
        double* Out = t.out_is_user ? userD : t.Out;
        const long long ldo = t.out_is_user ? ldd : t.ldo;
        const double* G = (t.sum_count == 1) ? t.sum_base : nullptr;
        if (t.sum_count > 1) return CHEB_DM_EUNSUPPORTED;  // the plan forces pre-formed sums
        if (t.ktiles == 0) {
            // product-free step (l = p - 1): Out = G
            if (!G) return CHEB_DM_EUNSUPPORTED;
            if (P->sym)  // only the tiles of G that touch the lower triangle exist (sliced_giant)
                unpad_copy_sym_kernel<<<P->num_sms * 4, 256, 0, st>>>(G, t.lds, P->N, Out, ldo, OZ_BM, OZ_BN);
            else
                unpad_copy_kernel<<<P->num_sms * 4, 256, 0, st>>>(G, t.lds, P->N, Out, ldo);
        } else {
            OzArgs oa;
            memset(&oa, 0, sizeof(oa));
            oa.alpha = t.alpha;
            oa.beta = t.C ? t.beta : 0.0;
            oa.C = t.C;
            oa.ldc = t.ldc;
            oa.G = G;
            oa.ldg = t.lds;
            oa.diag = t.diag_const;
            oa.Out = Out;
            oa.ldo = ldo;
            // Both factors are fetched K-major, i.e. the kernel forms (left) (right)^T.  Baby steps: T_l T_r^T, a one-off use of
            // the (rounding-level) asymmetry of T_r.  Giant steps and giant block: the accumulator (B_{l+1}, U_j) must be the
            // LEFT factor and the fixed multiplier Y = T_k the transposed one: with Y B^T an antisymmetric error component
            // between eigenvectors of Y with eigenvalues of opposite sign obeys e_l = 2 Y e_{l+1}^T - e_{l+2} and grows like
            // (c + sqrt(c^2 + 1))^l, c = sqrt|y_a y_b| (measured: 2e-7 at p = 32, 2e+4 at p = 64; reading A15);
            // with B Y^T every component follows the scalar recurrence and stays at the FP64 level.  Baby steps take the
            // higher-index operand as the left factor for the same reason (the serial pairing is such a recurrence in T_n).
            const int sa = oz_set_of_map(P, t.mapA), sb = oz_set_of_map(P, t.mapB);
            const bool swap = (kind != SLICED_BABY) || (sb > sa);
            s = oz_gemm(P, swap ? sb : sa, swap ? sa : sb, oa, P->sym, st);
            if (s != CHEB_DM_OK) return s;
        }
        ++P->last_launches;
        // is the result an operand of a later product?  T_n of the baby block: if a later baby product reads it, or n = k;
        // a giant-step accumulator B_l, l >= 1: always; U_{j+1}: by the next product of the chain
        if (!t.out_is_user) {
            const int m = (int)((t.Out - P->ws) / (long long)P->mat_elems);
            bool needed = (kind == SLICED_GIANT) || (kind == SLICED_CHAIN && lt + 1 < tt.ntl);
            if (kind == SLICED_BABY) {
                needed = (m == k - 1);
                for (int l2 = lt + 1; l2 < tt.ntl && !needed; ++l2) {
                    const Task& u = tt.h[(size_t)l2 * P->maxb];
                    needed = (u.mapA == m || u.mapB == m);
                }
            }
            if (needed) {
                s = oz_split(P, oz_set_of_matrix(P, m), t.Out, t.ldo, st);
                if (s != CHEB_DM_OK) return s;
                ++P->last_launches;
            }
        }
    }
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

// Baby block (T_1 is in place: front end).
cheb_dm_status_t sliced_baby(cheb_dm_plan_s* P, cudaStream_t st) {
    cheb_dm_status_t s = oz_split(P, 0, T_ptr(P, 0, 1), P->ld, st);  // T_1 = X
    if (s != CHEB_DM_OK) return s;
    ++P->last_launches;
    return sliced_table(P, P->baby, SLICED_BABY, nullptr, 0, st);
}

// Low-order sums (FP64; with symmetric tiles only the 128 x 64 tiles the products read: the product-free step, which
// needs a whole matrix, mirrors the rest) and the giant steps.
cheb_dm_status_t sliced_giant(cheb_dm_plan_s* P, double* userD, long long ldd, cudaStream_t st) {
    cheb_dm_status_t s = form_sums(P, 1, !P->sym, OZ_BM, OZ_BN, st);
    if (s != CHEB_DM_OK) return s;
    return sliced_table(P, P->giant, SLICED_GIANT, userD, ldd, st);
}

// The products of a fixed-mu solve on the sliced path.
cheb_dm_status_t run_products_sliced(cheb_dm_plan_s* P, double* userD, long long ldd, cudaStream_t st) {
    cheb_dm_status_t s = sliced_baby(P, st);
    if (s != CHEB_DM_OK) return s;
    return sliced_giant(P, userD, ldd, st);
}

}  // namespace

// =====================================================================================================
// C ABI
// =====================================================================================================
extern "C" {

const char* cheb_dm_strerror(cheb_dm_status_t s) {
    switch (s) {
        case CHEB_DM_OK: return "ok";
        case CHEB_DM_EINVAL: return "invalid argument";
        case CHEB_DM_EALLOC: return "workspace allocation failed";
        case CHEB_DM_ECUDA: return "CUDA error or no device";
        case CHEB_DM_ESTATE: return "call order violated";
        case CHEB_DM_EBOUNDS: return "bad spectral bounds";
        case CHEB_DM_EUNSUPPORTED: return "unsupported dtype or plan option";
        case CHEB_DM_ENOCONV: return "power-basis outer recursion would lose accuracy (use the Chebyshev outer recursion)";
        case CHEB_DM_ESIZE: return "N beyond CHEB_DM_STATIC_MAX_N = 8192, the fixed device scratch of cheb_dm_bounds_static";
    }
    return "unknown status";
}

cheb_dm_status_t cheb_dm_destroy(cheb_dm_plan_t P) {
    if (!P) return CHEB_DM_EINVAL;
    cudaFree(P->ws);
    cudaFree(P->costab);
    cudaFree(P->fn);
    cudaFree(P->c);
    cudaFree(P->gT);
    cudaFree(P->dT);
    cudaFree(P->Amat);
    cudaFree(P->tau);
    cudaFree(P->w);
    cudaFree(P->one);
    cudaFree(P->part);
    cudaFree(P->traces);
    cudaFree(P->gram_part);
    cudaFree(P->gram);
    cudaFree(P->sym_tiles);
    cudaFree(P->sym_panel_target);
    cudaFree(P->sc);
    cudaFree(P->maps);
    cudaFree(P->baby.d);
    cudaFree(P->giant.d);
    cudaFree(P->chain.d);
    cudaFree(P->flat.d);
    cudaFree(P->misc.d);
    cudaFree(P->counters);
    for (int i = 0; i < 2; ++i) {
        cudaFree(P->stage_H[i]);
        cudaFree(P->stage_D[i]);
        cudaFree(P->stage_tr[i]);
    }
    if (P->pipe_ready) {
        cudaStreamDestroy(P->s_in);
        cudaStreamDestroy(P->s_out);
        for (int i = 0; i < 2; ++i) {
            cudaEventDestroy(P->ev_in[i]);
            cudaEventDestroy(P->ev_comp[i]);
            cudaEventDestroy(P->ev_out[i]);
        }
    }
    cudaFree(P->oz_digits);
    cudaFree(P->oz_scale);
    cudaFree(P->oz_tiles[0]);
    cudaFree(P->oz_tiles[1]);
    cudaFree(P->trace_buf);
    for (int i = 0; i < TIMING_SLOTS; ++i) {
        if (P->ev0[i]) cudaEventDestroy(P->ev0[i]);
        if (P->ev1[i]) cudaEventDestroy(P->ev1[i]);
    }
    delete P;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_plan_ex(cheb_dm_plan_t* plan, int N, int M_terms, cheb_dm_dtype_t dtype,
                                 const cheb_dm_options_t* opts) {
    if (!plan || N < 1 || M_terms < 1) return CHEB_DM_EINVAL;
    if (dtype != CHEB_DM_F64) return CHEB_DM_EUNSUPPORTED;
    cheb_dm_options_t o;
    memset(&o, 0, sizeof(o));
    if (opts) o = *opts;
    if (o.k < 0 || o.p < 0) return CHEB_DM_EINVAL;
    if (o.outer != CHEB_DM_OUTER_CHEBYSHEV && o.outer != CHEB_DM_OUTER_POWER) return CHEB_DM_EINVAL;
    if (o.sched != CHEB_DM_SCHED_GROUPED && o.sched != CHEB_DM_SCHED_SERIAL) return CHEB_DM_EINVAL;
    if (o.pairing < CHEB_DM_PAIR_AUTO || o.pairing > CHEB_DM_PAIR_ALG1) return CHEB_DM_EINVAL;
    if (o.fuse_sums < 0 || o.fuse_sums > 2) return CHEB_DM_EINVAL;
    if (o.giant < 0 || o.giant > 2) return CHEB_DM_EINVAL;
    if (o.symmetric < 0 || o.symmetric > 2) return CHEB_DM_EINVAL;
    if (o.max_batch < 0 || o.max_batch > MAX_BATCH) return CHEB_DM_EINVAL;
    if ((o.ldh != 0 && o.ldh < N) || (o.ldd != 0 && o.ldd < N)) return CHEB_DM_EINVAL;
    if (o.moments < 0 || o.moments > 2 || o.host_slots < 0 || o.host_slots > 2) return CHEB_DM_EINVAL;
    if (o.sliced != 0 && (o.sliced < 2 || o.sliced > OZ_MAX_S || N > 65535)) return CHEB_DM_EINVAL;
    if (o.sliced_solve < 0 || o.sliced_solve > 1 || (o.sliced_solve && (o.max_batch > 1 || N > 65535))) return CHEB_DM_EINVAL;
    if (o.sliced_solve && o.sliced == 0) o.sliced = OZ_MAX_S;
    int k = o.k, p = o.p;
    if (k == 0 && p == 0) {
        k = 1;
        while ((long long)k * k < M_terms) ++k;  // k = ceil(sqrt(M))
        p = (M_terms + k - 1) / k;
    } else if (k == 0) {
        k = (M_terms + p - 1) / p;
    } else if (p == 0) {
        p = (M_terms + k - 1) / k;
    }
    if ((long long)k * p < M_terms) return CHEB_DM_EINVAL;

    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return CHEB_DM_ECUDA;
    CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    if (prop.major < 10) return CHEB_DM_ECUDA;  // the kernels are sm_100a only

    cheb_dm_plan_s* P = new (std::nothrow) cheb_dm_plan_s();
    if (!P) return CHEB_DM_EALLOC;
    P->N = N; P->M = M_terms; P->k = k; P->p = p;
    P->maxb = o.max_batch < 1 ? 1 : o.max_batch;
    P->opt = o; P->opt.k = k; P->opt.p = p; P->opt.max_batch = P->maxb;
    P->ldh = o.ldh ? o.ldh : N;
    P->ldd = o.ldd ? o.ldd : N;
    P->opt.ldh = (int)P->ldh; P->opt.ldd = (int)P->ldd;
    if (P->opt.pairing == CHEB_DM_PAIR_AUTO) P->opt.pairing = CHEB_DM_PAIR_BALANCED;
    P->device = dev; P->num_sms = prop.multiProcessorCount;
    int nq = 1;
    while (nq < 4 * M_terms) nq <<= 1;  // N_q = 2^ceil(log2(4M)) (cheb_dm.h)
    P->Nq = nq;
    P->sym = (o.symmetric != 1) ? 1 : 0;
    P->opt.symmetric = P->sym ? 2 : 1;
    {
        const char* env = getenv("CHEB_DM_SCALAR_SUMS");  // read here, never in a compute call
        P->scalar_sums = (env && env[0] == '1') ? 1 : 0;
    }
    choose_tile(P);
    P->panel_sym = (P->sym && P->BM % P->BN == 0) ? 1 : 0;
    P->ld = ((long long)N + 15) / 16 * 16;
    P->mat_elems = (((size_t)N * (size_t)P->ld) + 127) / 128 * 128;
    // Giant steps of single solves in the resident-multiplier kernel: N <= 512 (32 rows of T_k fit in shared memory),
    // operand maps with BK = 32 and 2-slab boxes (the 64x32 / 32x32 tile shapes), grouped scheduling, at least one
    // product, and k small enough for its coefficient staging area (k * GR_SUM_CHUNK doubles inside the idle TMA rings).
    P->resident = 0;
    P->res_tiles_m = P->res_tiles_n = ceil_div(N, 32);
    P->res_grid = P->sym ? (P->res_tiles_m * (P->res_tiles_m + 1)) / 2 : P->res_tiles_m * ceil_div(P->res_tiles_n, 2);
    P->res_smem = giant_resident_smem_bytes(ceil_div(N, GR_BK));
    if (o.giant != 1 && N <= 32 * GR_MAX_KTILES && p >= 2 && P->BK == GR_BK && P->box_slabs == 2 &&
        o.sched == CHEB_DM_SCHED_GROUPED && P->res_grid <= P->num_sms &&
        (long long)k * GR_SUM_CHUNK * 8 <= 2ll * GR_STAGES * GR_TILE_BYTES) {
        // (the attribute belongs to the kernel, not to the plan: opt in to the largest size any plan can ask for, or a later plan
        // for a smaller N would lower it under the feet of an earlier one)
        if (cudaFuncSetAttribute(giant_resident_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 giant_resident_smem_bytes(GR_MAX_KTILES)) == cudaSuccess) {
            int per_sm = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, giant_resident_kernel, GR_THREADS, P->res_smem) == cudaSuccess && per_sm >= 1)
                P->resident = 1;
        }
        cudaGetLastError();
    }
    P->opt.giant = P->resident ? 2 : 1;
    P->moments_on = (o.moments != 1) ? 1 : 0;
    P->opt.moments = P->moments_on ? 2 : 1;
    // a-5: fused (epilogue reads T_1..T_{k-1}: p (k-1) mat bytes per solve) while the baby blocks of the batch stay
    // L2-resident, pre-formed (form_sums_kernel: (ceil(p/16) (k-1) + p) mat bytes) once they do not.
    {
        int mode = o.fuse_sums;
        // (the epilogue warps of gemm_epi.cuh cannot gather k-1 tiles per item as fast as the consumers finish small-N
        // items: with those tile shapes the sums are always pre-formed)
        if (mode == 0) mode = (((double)k * (double)P->mat_elems * 8.0 * P->maxb > 96.0 * 1024 * 1024 || is_epi_tile(P->tile)) && k > 2 && p > 1) ? 2 : 1;
        if (o.sliced_solve) mode = 2;  // the sliced products add one pre-formed FP64 tile (any k, p: also G_l = g_l0 I for k = 1)
        P->preformed = (mode == 2) ? 1 : 0;
        P->opt.fuse_sums = mode;
    }
    if (P->resident && P->maxb == 1) {  // the resident kernel forms the sums itself (each CTA its own tiles) and parks them in G_l
        P->preformed = 1;
        P->opt.fuse_sums = 2;
    }
    if (P->resident && !P->preformed) {
        // a batch plan whose giant-step tasks gather the sums in their epilogues (fuse_sums = 1): the resident kernel reads
        // one pre-formed G tile per step, so single solves on such a plan (nbatch = 1) run in the generic kernel too
        P->resident = 0;
        P->opt.giant = 1;
    }
    const bool need_G = P->preformed || P->resident || P->moments_on;
    P->off_G = need_G ? k + NBUF : -1;
    P->off_U = (P->moments_on && p >= 3) ? k + NBUF + (need_G ? p : 0) : -1;
    P->nmat = k + NBUF + (need_G ? p : 0) + ((P->moments_on && p >= 3) ? p - 2 : 0);
    P->slot_elems = (size_t)P->nmat * P->mat_elems;
    P->map_flatA = k + NBUF;
    P->map_flatB = k + NBUF + (p - 1);
    P->nmaps_slot = k + NBUF + (P->moments_on ? 2 * (p - 1) : 0);
    P->ntrmat = k + ((P->moments_on && p >= 3) ? p - 2 : 0);
    {
        const long long nchunks = (long long)N * P->ld / 8;
        long long ctas = nchunks / 64;
        if (ctas > 2ll * P->num_sms) ctas = 2ll * P->num_sms;
        if (ctas < 1) ctas = 1;
        P->gram_ctas = (int)ctas;
        P->gram_passes = ceil_div(p > 1 ? p - 1 : 1, GRAM_BLK) * ceil_div(k > 1 ? k - 1 : 1, GRAM_BLK);
    }
    P->ws = nullptr; P->costab = P->fn = P->c = P->gT = P->dT = P->Amat = P->tau = P->w = P->one = P->part = nullptr;
    P->traces = P->gram_part = P->gram = nullptr;
    P->sym_tiles = nullptr; P->sym_panel_target = nullptr; P->sc = nullptr; P->maps = nullptr; P->counters = nullptr;
    P->have_coeffs = P->explicit_bounds = P->have_moments = P->computed = P->blocks_nb = 0;
    P->beta = P->mu = P->a = P->b = 0.0;
    P->last_launches = 0;
    P->work_next = 0;
    for (int i = 0; i < 2; ++i) P->stage_H[i] = P->stage_D[i] = P->stage_tr[i] = nullptr;
    P->pipe_ready = 0;
    P->n_async = 0;
    P->timing = 0; P->ev_count = 0;
    P->trace_buf = nullptr; P->trace_on = 0; P->trace_nb = 1;
    P->opt.sliced = o.sliced;
    P->oz_S = o.sliced; P->oz_solve = o.sliced_solve; P->oz_nsets = 0; P->oz_kpad = ((long long)N + OZ_BK - 1) / OZ_BK * OZ_BK; P->oz_digits = nullptr; P->oz_scale = nullptr; P->oz_tiles[0] = P->oz_tiles[1] = nullptr;
    for (int i = 0; i < TIMING_SLOTS; ++i) P->ev0[i] = P->ev1[i] = nullptr;

    const size_t kp = (size_t)k * p, B = (size_t)P->maxb;
    P->ws_bytes = sizeof(double) * P->slot_elems * B;
    bool ok = true;
    ok = ok && cudaMalloc(&P->ws, P->ws_bytes) == cudaSuccess;
    ok = ok && cudaMalloc(&P->costab, sizeof(double) * 4 * nq) == cudaSuccess;
    ok = ok && cudaMalloc(&P->fn, sizeof(double) * nq * B) == cudaSuccess;
    ok = ok && cudaMalloc(&P->c, sizeof(double) * kp * B) == cudaSuccess;
    ok = ok && cudaMalloc(&P->gT, sizeof(double) * kp * B) == cudaSuccess;
    ok = ok && cudaMalloc(&P->dT, sizeof(double) * kp * B) == cudaSuccess;
    ok = ok && cudaMalloc(&P->Amat, sizeof(double) * p * p) == cudaSuccess;
    ok = ok && cudaMalloc(&P->tau, sizeof(double) * kp * B) == cudaSuccess;
    ok = ok && cudaMalloc(&P->w, sizeof(double) * nq * B) == cudaSuccess;
    ok = ok && cudaMalloc(&P->sc, sizeof(DevScalars) * B) == cudaSuccess;
    ok = ok && cudaMalloc(&P->one, sizeof(double)) == cudaSuccess;
    const size_t gram_part_elems = B * P->gram_passes * P->gram_ctas * (size_t)(GRAM_BLK * GRAM_BLK);
    if (P->moments_on) {
        ok = ok && cudaMalloc(&P->traces, sizeof(double) * B * P->ntrmat) == cudaSuccess;
        ok = ok && cudaMalloc(&P->gram_part, sizeof(double) * gram_part_elems) == cudaSuccess;
        ok = ok && cudaMalloc(&P->gram, sizeof(double) * B * (kp + 1)) == cudaSuccess;
    }
    {
        int per_sm = 0;
        ok = ok && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, front_end_kernel, 512, 0) == cudaSuccess && per_sm >= 1;
        P->front_max_grid = per_sm * P->num_sms;
        if (P->front_max_grid > 4 * P->num_sms) P->front_max_grid = 4 * P->num_sms;
        ok = ok && P->front_max_grid >= P->maxb;
        ok = ok && cudaMalloc(&P->part, sizeof(double) * 2 * (P->front_max_grid > 0 ? P->front_max_grid : 1)) == cudaSuccess;
    }
    ok = ok && cudaMalloc(&P->maps, sizeof(CUtensorMap) * P->nmaps_slot * B) == cudaSuccess;
    for (int i = 0; i < TIMING_SLOTS && ok; ++i)
        ok = cudaEventCreate(&P->ev0[i]) == cudaSuccess && cudaEventCreate(&P->ev1[i]) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        cheb_dm_destroy(P);
        return CHEB_DM_EALLOC;
    }
    P->ws_bytes += sizeof(double) * (4 * (size_t)nq + B * (2 * nq + 4 * kp) + (size_t)p * p + (P->moments_on ? gram_part_elems : 0));

    cheb_dm_status_t st = CHEB_DM_OK;
    do {
        if (prepare_gemm(P) != CHEB_DM_OK) { cudaGetLastError(); st = CHEB_DM_ECUDA; break; }
        if (cudaMemset(P->ws, 0, sizeof(double) * P->slot_elems * B) != cudaSuccess) { st = CHEB_DM_ECUDA; break; }
        cudaMemset(P->dT, 0, sizeof(double) * kp * B);
        cudaMemset(P->gT, 0, sizeof(double) * kp * B);
        cudaMemset(P->c, 0, sizeof(double) * kp * B);
        cudaMemset(P->tau, 0, sizeof(double) * kp * B);
        cudaMemset(P->sc, 0, sizeof(DevScalars) * B);
        {
            const double one = 1.0;
            cudaMemcpy(P->one, &one, sizeof(double), cudaMemcpyHostToDevice);
        }
        std::vector<double> tab, A;
        build_costab(nq, tab);
        build_Amat(p, A);
        if (cudaMemcpy(P->costab, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(P->Amat, A.data(), sizeof(double) * A.size(), cudaMemcpyHostToDevice) != cudaSuccess) {
            st = CHEB_DM_ECUDA;
            break;
        }
        {
            const int tn_ = ceil_div(N, P->BN), tm_ = ceil_div(N, P->BM);
            // Work item -> tile of a symmetric task.  Column-panel-major (a panel's tiles are consecutive: with the per-panel
            // dependencies the next level's first panels are ready early) while a matrix fits the L2 several times over; for
            // larger matrices in bands of 16 column panels, row block by row block inside a band: a wave of ~148 tiles then
            // touches ~9 A row blocks and 16 B column panels instead of every A row block (measured at N = 5000 with 64x64
            // tiles, panel-major: 4.5 GB of DRAM reads per product against 0.6 GB of operands).
            std::vector<short2> tl;
            const bool banded = (double)N * (double)P->ld * 8.0 > 48.0 * 1024 * 1024;
            const int band = banded ? 16 : 1;
            for (int b0 = 0; b0 < tn_; b0 += band) {
                if (!banded) {
                    for (int tm = sym_tm0(b0, P->BM, P->BN); tm < tm_; ++tm) tl.push_back(make_short2((short)tm, (short)b0));
                } else {
                    for (int tm = 0; tm < tm_; ++tm)
                        for (int tn = b0; tn < tn_ && tn < b0 + band; ++tn)
                            if (tm >= sym_tm0(tn, P->BM, P->BN)) tl.push_back(make_short2((short)tm, (short)tn));
                }
            }
            if ((int)tl.size() != sym_items(N, P->BM, P->BN)) { st = CHEB_DM_EINVAL; break; }
            if (cudaMalloc(&P->sym_tiles, sizeof(short2) * tl.size()) != cudaSuccess) { cudaGetLastError(); st = CHEB_DM_EALLOC; break; }
            if (cudaMemcpy(P->sym_tiles, tl.data(), sizeof(short2) * tl.size(), cudaMemcpyHostToDevice) != cudaSuccess) { st = CHEB_DM_ECUDA; break; }
            // column panel q of a symmetric result is written by the work items of panel q and, mirrored, by the work items
            // (tm, tn != q) of the row block(s) tm whose rows cross the panel's columns: q in [tm R, tm R + R), R = BM / BN
            std::vector<int> tg(tn_, 0);
            if (P->panel_sym) {
                const int R = P->BM / P->BN;
                for (int tn = 0; tn < tn_; ++tn)
                    for (int tm = sym_tm0(tn, P->BM, P->BN); tm < tm_; ++tm) {
                        ++tg[tn];
                        for (int u = 0; u < R; ++u) {
                            const int q = tm * R + u;
                            if (q != tn && q < tn_) ++tg[q];
                        }
                    }
            }
            if (cudaMalloc(&P->sym_panel_target, sizeof(int) * tg.size()) != cudaSuccess) { cudaGetLastError(); st = CHEB_DM_EALLOC; break; }
            if (cudaMemcpy(P->sym_panel_target, tg.data(), sizeof(int) * tg.size(), cudaMemcpyHostToDevice) != cudaSuccess) { st = CHEB_DM_ECUDA; break; }
        }
        st = encode_maps(P);
        if (st != CHEB_DM_OK) break;
        build_tables(P);
        P->panel_stride = ceil_div(N, 16);  // >= the number of column panels of every kernel (narrowest panel: 16)
        TaskTable* tabs[5] = {&P->baby, &P->giant, &P->chain, &P->flat, &P->misc};
        size_t off = 1;  // [0] = sticky error flag
        int total_tasks = 0, trace_off = 0;
        for (int t = 0; t < 5; ++t) total_tasks += (int)tabs[t]->h.size();
        P->nwork = total_tasks + 8;
        off += P->nwork;
        for (int t = 0; t < 5; ++t) {
            TaskTable* tt = tabs[t];
            tt->ctr_task_off = (int)off;
            off += tt->h.size();
            tt->ctr_panel_off = (int)off;
            off += tt->h.size() * (size_t)P->panel_stride;
            tt->trace_base = trace_off;
            trace_off += tt->ntl * tt->items_per_task * P->maxb;
        }
        P->trace_res_base = trace_off;
        P->trace_total = trace_off + P->p * P->res_tiles_m * P->res_tiles_n;
        P->counters_ints = off;
        if (cudaMalloc(&P->counters, sizeof(int) * P->counters_ints) != cudaSuccess) { cudaGetLastError(); st = CHEB_DM_EALLOC; break; }
        if (cudaMemset(P->counters, 0, sizeof(int) * P->counters_ints) != cudaSuccess) { st = CHEB_DM_ECUDA; break; }
        for (int t = 0; t < 5 && st == CHEB_DM_OK; ++t) {
            TaskTable* tt = tabs[t];
            if (tt->h.empty()) continue;
            if (cudaMalloc(&tt->d, sizeof(Task) * tt->h.size()) != cudaSuccess) { cudaGetLastError(); st = CHEB_DM_EALLOC; break; }
            if (cudaMemcpy(tt->d, tt->h.data(), sizeof(Task) * tt->h.size(), cudaMemcpyHostToDevice) != cudaSuccess) st = CHEB_DM_ECUDA;
        }
        if (st != CHEB_DM_OK) break;
        if (o.host_slots > 0) {
            st = ensure_staging(P, o.host_slots);
            if (st != CHEB_DM_OK) break;
        }
        if (P->oz_S > 0) {
            st = prepare_sliced(P);
            if (st != CHEB_DM_OK) break;
        }
        if (cudaDeviceSynchronize() != cudaSuccess) { st = CHEB_DM_ECUDA; break; }
    } while (0);
    if (st != CHEB_DM_OK) {
        cheb_dm_destroy(P);
        return st;
    }
    *plan = P;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_plan(cheb_dm_plan_t* plan, int N, int M_terms, cheb_dm_dtype_t dtype) {
    return cheb_dm_plan_ex(plan, N, M_terms, dtype, nullptr);
}

cheb_dm_status_t cheb_dm_coeffs(cheb_dm_plan_t P, double beta, double mu, const double* bounds) {
    if (!P) return CHEB_DM_EINVAL;
    if (!isfinite(beta) || !isfinite(mu) || !(beta > 0.0)) return CHEB_DM_EINVAL;
    if (bounds) {
        if (!isfinite(bounds[0]) || !isfinite(bounds[1]) || !(bounds[1] > bounds[0])) return CHEB_DM_EBOUNDS;
    }
    // The blocks a cheb_dm_moments / cheb_dm_solve call left in the workspace are polynomials of X = X(a, b): new bounds (or
    // a new bounds mode) make them stale -- cheb_dm_assemble / cheb_dm_solve_mu then return ESTATE instead of a D for the old
    // scaling.  A new beta or mu alone keeps them.
    const int was_explicit = P->explicit_bounds;
    if ((bounds != nullptr) != (was_explicit != 0) || (bounds && (bounds[0] != P->a || bounds[1] != P->b))) {
        P->blocks_nb = 0;
        P->have_moments = 0;
    }
    if (bounds) {
        P->a = bounds[0];
        P->b = bounds[1];
        P->explicit_bounds = 1;
    } else {
        P->explicit_bounds = 0;
    }
    P->beta = beta;
    P->mu = mu;
    P->have_coeffs = 1;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_get_options(cheb_dm_plan_t P, cheb_dm_options_t* opts_out) {
    if (!P || !opts_out) return CHEB_DM_EINVAL;
    *opts_out = P->opt;
    opts_out->tile = P->tile;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_get_kp(cheb_dm_plan_t P, int* k_out, int* p_out) {
    if (!P || !k_out || !p_out) return CHEB_DM_EINVAL;
    *k_out = P->k;
    *p_out = P->p;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_workspace_bytes(cheb_dm_plan_t P, size_t* bytes_out) {
    if (!P || !bytes_out) return CHEB_DM_EINVAL;
    *bytes_out = P->ws_bytes;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_last_launch_count(cheb_dm_plan_t P, int* launches_out) {
    if (!P || !launches_out) return CHEB_DM_EINVAL;
    *launches_out = P->last_launches;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_flops_per_compute(cheb_dm_plan_t P, double* flops_out) {
    if (!P || !flops_out) return CHEB_DM_EINVAL;
    *flops_out = P->flops_per_compute;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_sliced_ops_per_compute(cheb_dm_plan_t P, double* ops_out) {
    if (!P || !ops_out) return CHEB_DM_EINVAL;
    if (!P->oz_solve) return CHEB_DM_EUNSUPPORTED;
    const double S = (double)P->oz_S;
    const double products = (double)P->baby.ntl + (double)(P->p > 1 ? P->p - 1 : 0);
    *ops_out = products * (S * (S + 1.0) / 2.0) * 2.0 * (double)P->oz_ntiles[P->sym ? 1 : 0] * OZ_BM * OZ_BN * (double)P->oz_kpad;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_flops_per_solve(cheb_dm_plan_t P, double* flops_out) {
    if (!P || !flops_out) return CHEB_DM_EINVAL;
    if (!P->moments_on) return CHEB_DM_EUNSUPPORTED;
    *flops_out = P->flops_per_solve;
    return CHEB_DM_OK;
}

// ------------------------------------------------------------------------------------------------------
// fixed-mu solves
// ------------------------------------------------------------------------------------------------------
cheb_dm_status_t cheb_dm_compute_batch(cheb_dm_plan_t P, int nbatch, const double* const* dH, double* const* dD, const double* mu,
                                       void* cuda_stream) {
    if (!P || !batch_args_ok(P, nbatch, dH, dD, mu)) return CHEB_DM_EINVAL;
    if (!P->have_coeffs) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    return compute_impl(P, nbatch, dH, P->ldh, dD, P->ldd, mu, (cudaStream_t)cuda_stream);
}

cheb_dm_status_t cheb_dm_compute(cheb_dm_plan_t P, const double* dH, double* dD, void* cuda_stream) {
    if (!P || !dH || !dD || dH == dD) return CHEB_DM_EINVAL;
    return cheb_dm_compute_batch(P, 1, &dH, &dD, nullptr, cuda_stream);
}

cheb_dm_status_t cheb_dm_compute_batch_host_async(cheb_dm_plan_t P, int nbatch, const double* const* hH, double* const* hD,
                                                  double* h_trace, const double* mu, void* cuda_stream) {
    if (!P || !batch_args_ok(P, nbatch, hH, hD, mu)) return CHEB_DM_EINVAL;
    if (!P->have_coeffs) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cheb_dm_status_t s = ensure_staging(P, 2);
    if (s != CHEB_DM_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t elems = (size_t)P->N * P->N, bytes = sizeof(double) * elems;
    const int set = (int)(P->n_async & 1);
    const double* sH[MAX_BATCH];
    double* sD[MAX_BATCH];
    for (int i = 0; i < nbatch; ++i) {
        sH[i] = P->stage_H[set] + (size_t)i * elems;
        sD[i] = P->stage_D[set] + (size_t)i * elems;
    }
    // H2D of this call: the set's previous occupant (call n-2) must have been consumed by its kernels
    if (P->n_async >= 2) CUDA_TRY(cudaStreamWaitEvent(P->s_in, P->ev_comp[set], 0));
    for (int i = 0; i < nbatch; ++i) CUDA_TRY(cudaMemcpyAsync((void*)sH[i], hH[i], bytes, cudaMemcpyHostToDevice, P->s_in));
    CUDA_TRY(cudaEventRecord(P->ev_in[set], P->s_in));
    // kernels, in call order on the caller's stream: need this call's H and the set's D / tr copied out (call n-2)
    CUDA_TRY(cudaStreamWaitEvent(st, P->ev_in[set], 0));
    if (P->n_async >= 2) CUDA_TRY(cudaStreamWaitEvent(st, P->ev_out[set], 0));
    s = compute_impl(P, nbatch, sH, P->N, sD, P->N, mu, st);
    if (s != CHEB_DM_OK) return s;
    if (h_trace) {
        s = trace_impl(P, nbatch, sD, P->N, P->stage_tr[set], st);
        if (s != CHEB_DM_OK) return s;
        ++P->last_launches;
    }
    CUDA_TRY(cudaEventRecord(P->ev_comp[set], st));
    // D2H of this call
    CUDA_TRY(cudaStreamWaitEvent(P->s_out, P->ev_comp[set], 0));
    if (h_trace) CUDA_TRY(cudaMemcpyAsync(h_trace, P->stage_tr[set], sizeof(double) * nbatch, cudaMemcpyDeviceToHost, P->s_out));
    for (int i = 0; i < nbatch; ++i) CUDA_TRY(cudaMemcpyAsync(hD[i], sD[i], bytes, cudaMemcpyDeviceToHost, P->s_out));
    CUDA_TRY(cudaEventRecord(P->ev_out[set], P->s_out));
    ++P->n_async;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_compute_batch_host(cheb_dm_plan_t P, int nbatch, const double* const* hH, double* const* hD, double* h_trace,
                                            const double* mu, void* cuda_stream) {
    if (!P || !batch_args_ok(P, nbatch, hH, hD, mu)) return CHEB_DM_EINVAL;
    if (!P->have_coeffs) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cheb_dm_status_t s = ensure_staging(P, 1);
    if (s != CHEB_DM_OK) return s;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t elems = (size_t)P->N * P->N, bytes = sizeof(double) * elems;
    const double* sH[MAX_BATCH];
    double* sD[MAX_BATCH];
    for (int i = 0; i < nbatch; ++i) {
        sH[i] = P->stage_H[0] + (size_t)i * elems;
        sD[i] = P->stage_D[0] + (size_t)i * elems;
        CUDA_TRY(cudaMemcpyAsync((void*)sH[i], hH[i], bytes, cudaMemcpyHostToDevice, st));
    }
    s = compute_impl(P, nbatch, sH, P->N, sD, P->N, mu, st);
    if (s != CHEB_DM_OK) return s;
    if (h_trace) {
        s = trace_impl(P, nbatch, sD, P->N, P->stage_tr[0], st);
        if (s != CHEB_DM_OK) return s;
        ++P->last_launches;
        CUDA_TRY(cudaMemcpyAsync(h_trace, P->stage_tr[0], sizeof(double) * nbatch, cudaMemcpyDeviceToHost, st));
    }
    for (int i = 0; i < nbatch; ++i) CUDA_TRY(cudaMemcpyAsync(hD[i], sD[i], bytes, cudaMemcpyDeviceToHost, st));
    return cheb_dm_check(P, cuda_stream);  // synchronises the stream
}

cheb_dm_status_t cheb_dm_compute_host(cheb_dm_plan_t P, const double* hH, double* hD, double* h_trace, void* cuda_stream) {
    if (!P || !hH || !hD || hH == hD) return CHEB_DM_EINVAL;
    return cheb_dm_compute_batch_host(P, 1, &hH, &hD, h_trace, nullptr, cuda_stream);
}

cheb_dm_status_t cheb_dm_compute_host_async(cheb_dm_plan_t P, const double* hH, double* hD, double* h_trace, void* cuda_stream) {
    if (!P || !hH || !hD || hH == hD) return CHEB_DM_EINVAL;
    return cheb_dm_compute_batch_host_async(P, 1, &hH, &hD, h_trace, nullptr, cuda_stream);
}

cheb_dm_status_t cheb_dm_wait(cheb_dm_plan_t P, void* cuda_stream) {
    if (!P) return CHEB_DM_EINVAL;
    if (P->pipe_ready) {
        CUDA_TRY(cudaStreamSynchronize(P->s_in));
        CUDA_TRY(cudaStreamSynchronize(P->s_out));
    }
    return cheb_dm_check(P, cuda_stream);
}

cheb_dm_status_t cheb_dm_check(cheb_dm_plan_t P, void* cuda_stream) {
    if (!P) return CHEB_DM_EINVAL;
    if (!P->computed) return CHEB_DM_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int flag = 0;
    std::vector<DevScalars> h((size_t)P->maxb);
    CUDA_TRY(cudaMemcpyAsync(&flag, P->counters, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(h.data(), P->sc, sizeof(DevScalars) * P->maxb, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    bool bad = false, noconv = false;
    for (int s = 0; s < P->maxb; ++s) {
        bad = bad || h[s].bad_bounds;
        noconv = noconv || h[s].noconv;
    }
    if (flag) CUDA_TRY(cudaMemsetAsync(P->counters, 0, sizeof(int), st));  // the flags are sticky until reported here
    if (bad || noconv)
        for (int s = 0; s < P->maxb; ++s)
            if (h[s].bad_bounds || h[s].noconv) CUDA_TRY(cudaMemsetAsync(&P->sc[s].bad_bounds, 0, 2 * sizeof(int), st));
    if (flag) return CHEB_DM_ECUDA;
    if (bad) return CHEB_DM_EBOUNDS;
    if (noconv) return CHEB_DM_ENOCONV;
    return CHEB_DM_OK;
}

// ------------------------------------------------------------------------------------------------------
// moments, mu search, mu-inclusive solve
// ------------------------------------------------------------------------------------------------------
cheb_dm_status_t cheb_dm_moments(cheb_dm_plan_t P, const double* dH, double* tau_host, void* cuda_stream) {
    if (!P || !dH) return CHEB_DM_EINVAL;
    if (!P->moments_on) return CHEB_DM_EUNSUPPORTED;
    if (!P->have_coeffs) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    P->last_launches = 0;
    cheb_dm_status_t s = front_end(P, 1, &dH, P->ldh, nullptr, 1, 0, 0, st);  // counters reset, bounds + rescale
    if (s != CHEB_DM_OK) return s;
    s = blocks_and_moments(P, 1, st);
    if (s != CHEB_DM_OK) return s;
    P->have_moments = 1;
    P->blocks_nb = 1;
    P->computed = 1;
    if (tau_host) {
        CUDA_TRY(cudaMemcpyAsync(tau_host, P->tau, sizeof(double) * (size_t)P->k * P->p, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
    }
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_solve_mu(cheb_dm_plan_t P, double beta, double n_occ, int iters, double* mu_out, void* cuda_stream) {
    if (!P || !mu_out || iters < 1 || !isfinite(beta) || !(beta > 0.0) || !isfinite(n_occ)) return CHEB_DM_EINVAL;
    if (!P->have_moments) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cheb_dm_status_t s = bisect(P, 1, beta, &n_occ, iters, st);
    if (s != CHEB_DM_OK) return s;
    DevScalars h;
    CUDA_TRY(cudaMemcpyAsync(&h, P->sc, sizeof(h), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (h.bad_bounds) return CHEB_DM_EBOUNDS;
    *mu_out = h.mu;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_solve_batch(cheb_dm_plan_t P, int nbatch, const double* const* dH, const double* n_occ, int iters,
                                     double* const* dD, double* mu_out, void* cuda_stream) {
    if (!P || !n_occ || iters < 1 || !batch_args_ok(P, nbatch, dH, dD, nullptr)) return CHEB_DM_EINVAL;
    for (int s = 0; s < nbatch; ++s)
        if (!isfinite(n_occ[s])) return CHEB_DM_EINVAL;
    if (!P->moments_on) return CHEB_DM_EUNSUPPORTED;
    if (!P->have_coeffs) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    P->last_launches = 0;
    cheb_dm_status_t s = front_end(P, nbatch, dH, P->ldh, nullptr, 1, 0, 0, st);
    if (s != CHEB_DM_OK) return s;
    const int slot = (int)(P->ev_count % TIMING_SLOTS);
    if (P->timing) CUDA_TRY(cudaEventRecord(P->ev0[slot], st));
    s = blocks_and_moments(P, nbatch, st);
    if (s != CHEB_DM_OK) return s;
    s = bisect(P, nbatch, P->beta, n_occ, iters, st);
    if (s != CHEB_DM_OK) return s;
    s = assemble_impl(P, nbatch, nullptr, 1, dD, P->ldd, st);
    if (s != CHEB_DM_OK) return s;
    if (P->timing) {
        CUDA_TRY(cudaEventRecord(P->ev1[slot], st));
        ++P->ev_count;
    }
    P->computed = 1;
    P->have_moments = (nbatch == 1);
    P->blocks_nb = nbatch;
    if (mu_out) {
        std::vector<DevScalars> h((size_t)nbatch);
        CUDA_TRY(cudaMemcpyAsync(h.data(), P->sc, sizeof(DevScalars) * nbatch, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        for (int i = 0; i < nbatch; ++i)
            if (h[i].bad_bounds) return CHEB_DM_EBOUNDS;
        for (int i = 0; i < nbatch; ++i) mu_out[i] = h[i].mu;
    }
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_solve(cheb_dm_plan_t P, const double* dH, double n_occ, int iters, double* dD, double* mu_out,
                               void* cuda_stream) {
    if (!P || !dH || !dD || dH == dD) return CHEB_DM_EINVAL;
    return cheb_dm_solve_batch(P, 1, &dH, &n_occ, iters, &dD, mu_out, cuda_stream);
}

cheb_dm_status_t cheb_dm_assemble(cheb_dm_plan_t P, int nbatch, const double* mu, double* const* dD, void* cuda_stream) {
    if (!P || !mu || !dD || nbatch < 1 || nbatch > P->maxb) return CHEB_DM_EINVAL;
    for (int s = 0; s < nbatch; ++s)
        if (!dD[s] || !isfinite(mu[s])) return CHEB_DM_EINVAL;
    if (!P->moments_on) return CHEB_DM_EUNSUPPORTED;
    if (!P->have_coeffs || P->blocks_nb != nbatch) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    P->last_launches = 0;
    return assemble_impl(P, nbatch, mu, 0, dD, P->ldd, (cudaStream_t)cuda_stream);
}

// ------------------------------------------------------------------------------------------------------
// trace, getters
// ------------------------------------------------------------------------------------------------------
cheb_dm_status_t cheb_dm_trace_batch(cheb_dm_plan_t P, int nbatch, const double* const* dD, double* trace_out, void* cuda_stream) {
    if (!P || !dD || !trace_out || nbatch < 1 || nbatch > MAX_BATCH) return CHEB_DM_EINVAL;
    for (int s = 0; s < nbatch; ++s)
        if (!dD[s]) return CHEB_DM_EINVAL;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    return trace_impl(P, nbatch, dD, P->ldd, trace_out, (cudaStream_t)cuda_stream);
}

cheb_dm_status_t cheb_dm_trace(cheb_dm_plan_t P, const double* dD, double* trace_out, void* cuda_stream) {
    if (!P || !dD || !trace_out) return CHEB_DM_EINVAL;
    return cheb_dm_trace_batch(P, 1, &dD, trace_out, cuda_stream);
}

cheb_dm_status_t cheb_dm_get_scalars(cheb_dm_plan_t P, int slot, double* out4, void* cuda_stream) {
    if (!P || !out4 || slot < 0 || slot >= P->maxb) return CHEB_DM_EINVAL;
    if (!P->computed) return CHEB_DM_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DevScalars h;
    CUDA_TRY(cudaMemcpyAsync(&h, P->sc + slot, sizeof(h), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (h.bad_bounds || !isfinite(h.a) || !isfinite(h.b)) return CHEB_DM_EBOUNDS;
    out4[0] = h.a;
    out4[1] = h.b;
    out4[2] = h.mu;
    out4[3] = h.ne;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_get_bounds(cheb_dm_plan_t P, double* bounds_out, void* cuda_stream) {
    if (!P || !bounds_out) return CHEB_DM_EINVAL;
    double v[4];
    cheb_dm_status_t s = cheb_dm_get_scalars(P, 0, v, cuda_stream);
    if (s != CHEB_DM_OK) return s;
    bounds_out[0] = v[0];
    bounds_out[1] = v[1];
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_get_coeffs(cheb_dm_plan_t P, double* c_out, double* g_out, double* d_out, void* cuda_stream) {
    if (!P) return CHEB_DM_EINVAL;
    if (!P->computed) return CHEB_DM_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int k = P->k, p = P->p;
    const size_t kp = (size_t)k * p;
    std::vector<double> tmp(kp);
    if (c_out) CUDA_TRY(cudaMemcpyAsync(c_out, P->c, sizeof(double) * kp, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    for (int which = 0; which < 2; ++which) {
        double* out = which == 0 ? g_out : d_out;
        if (!out) continue;
        CUDA_TRY(cudaMemcpyAsync(tmp.data(), which == 0 ? P->gT : P->dT, sizeof(double) * kp, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
        for (int l = 0; l < p; ++l)
            for (int i = 0; i < k; ++i) out[(size_t)i * p + l] = tmp[(size_t)l * k + i];  // device layout is [l][i]
    }
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_get_T(cheb_dm_plan_t P, int n, double* dOut, void* cuda_stream) {
    if (!P || !dOut || n < 1 || n > P->k) return CHEB_DM_EINVAL;
    if (!P->computed) return CHEB_DM_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    unpad_copy_kernel<<<P->num_sms * 4, 256, 0, st>>>(T_ptr(P, 0, n), P->ld, P->N, dOut, P->N);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaStreamSynchronize(st));
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_product(cheb_dm_plan_t P, double alpha, const double* dA, const double* dB, double beta,
                                 const double* dC, double* dOut, void* cuda_stream) {
    if (!P || !dA || !dB || !dOut) return CHEB_DM_EINVAL;
    if (dOut == dA || dOut == dB) return CHEB_DM_EINVAL;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // operands go through the TMA-described workspace buffers (this also handles odd N)
    pad_copy_kernel<<<P->num_sms * 4, 256, 0, st>>>(dA, P->N, P->N, buf_ptr(P, 0, 0), P->ld);
    pad_copy_kernel<<<P->num_sms * 4, 256, 0, st>>>(dB, P->N, P->N, buf_ptr(P, 0, 1), P->ld);
    Task t = P->misc.h[0];
    t.alpha = alpha;
    t.beta = beta;
    t.C = dC;
    t.ldc = P->N;
    CUDA_TRY(cudaMemcpyAsync(P->misc.d, &t, sizeof(Task), cudaMemcpyHostToDevice, st));
    const int save = P->last_launches, wsave = P->work_next;
    P->work_next = P->nwork - 1;  // the last work counter is reserved for this call
    CUDA_TRY(cudaMemsetAsync(P->counters + 1 + P->work_next, 0, sizeof(int), st));
    cheb_dm_status_t s = launch_tasks(P, P->misc, 0, 1, 1, 0, &dOut, P->N, st);
    P->last_launches = save;
    P->work_next = wsave;
    // the pageable-source copy above is staged by the runtime before it returns, so `t` may go out of scope
    return s;
}

cheb_dm_status_t cheb_dm_product_sliced(cheb_dm_plan_t P, double alpha, const double* dA, const double* dB, double beta,
                                        const double* dC, double* dOut, int symmetric, void* cuda_stream) {
    if (!P || !dA || !dB || !dOut) return CHEB_DM_EINVAL;
    if (dOut == dA || dOut == dB) return CHEB_DM_EINVAL;
    if (P->oz_S < 2) return CHEB_DM_EUNSUPPORTED;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int N = P->N;
    const int same = (dA == dB) ? 1 : 0;
    const int setA = P->oz_nsets - 2, setB = same ? setA : P->oz_nsets - 1;
    cheb_dm_status_t s = oz_split(P, setA, dA, N, st);
    if (s == CHEB_DM_OK && !same) s = oz_split(P, setB, dB, N, st);
    if (s != CHEB_DM_OK) return s;
    OzArgs oa;
    memset(&oa, 0, sizeof(oa));
    oa.alpha = alpha;
    oa.beta = dC ? beta : 0.0;
    oa.C = dC;
    oa.ldc = N;
    oa.Out = dOut;
    oa.ldo = N;
    return oz_gemm(P, setA, setB, oa, symmetric, st);
}

// ------------------------------------------------------------------------------------------------------
// tracing and measurement support
// ------------------------------------------------------------------------------------------------------
cheb_dm_status_t cheb_dm_set_trace(cheb_dm_plan_t P, int enable) {
    if (!P) return CHEB_DM_EINVAL;
    if (enable && !P->trace_buf) {
        const size_t n = (size_t)P->trace_total;
        if (cudaMalloc(&P->trace_buf, sizeof(TraceRec) * n) != cudaSuccess) {
            cudaGetLastError();
            P->trace_buf = nullptr;
            return CHEB_DM_EALLOC;
        }
        CUDA_TRY(cudaMemset(P->trace_buf, 0, sizeof(TraceRec) * n));
    }
    P->trace_on = enable ? 1 : 0;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_get_trace(cheb_dm_plan_t P, cheb_dm_trace_rec_t* out, int max_records, int* count_out) {
    if (!P || !out || !count_out || max_records < 0) return CHEB_DM_EINVAL;
    if (!P->trace_buf) return CHEB_DM_ESTATE;
    static_assert(sizeof(cheb_dm_trace_rec_t) == sizeof(TraceRec), "trace record layout");
    CUDA_TRY(cudaDeviceSynchronize());
    int n = 0;
    // baby-step items, then the giant steps (generic kernel items or resident-kernel tiles), of the nb matrices of the
    // last traced call, in claim order (level by level, matrix by matrix)
    const int tnb = P->trace_nb > 0 ? P->trace_nb : 1;
    const bool res = P->resident && tnb == 1;
    const TaskTable* tabs[2] = {&P->baby, res ? nullptr : &P->giant};
    for (int t = 0; t < 2; ++t) {
        if (!tabs[t]) continue;
        int m = tabs[t]->ntl * tabs[t]->items_per_task * tnb;
        if (m > max_records - n) m = max_records - n;
        if (m > 0) CUDA_TRY(cudaMemcpy(out + n, P->trace_buf + tabs[t]->trace_base, sizeof(TraceRec) * (size_t)m, cudaMemcpyDeviceToHost));
        n += m > 0 ? m : 0;
    }
    if (res) {
        const int m = P->p * P->res_tiles_m * P->res_tiles_n;
        std::vector<TraceRec> tmp((size_t)m);
        CUDA_TRY(cudaMemcpy(tmp.data(), P->trace_buf + P->trace_res_base, sizeof(TraceRec) * (size_t)m, cudaMemcpyDeviceToHost));
        for (int i = 0; i < m && n < max_records; ++i)
            if (tmp[i].t_done != 0) {  // tiles above the diagonal are not work items in symmetric mode
                memcpy(out + n, &tmp[i], sizeof(TraceRec));
                ++n;
            }
    }
    *count_out = n;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_set_timing(cheb_dm_plan_t P, int enable) {
    if (!P) return CHEB_DM_EINVAL;
    P->timing = enable ? 1 : 0;
    P->ev_count = 0;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_product_ms(cheb_dm_plan_t P, int* count_out, double* total_ms_out) {
    if (!P || !count_out || !total_ms_out) return CHEB_DM_EINVAL;
    if (!P->timing || P->ev_count < 1) return CHEB_DM_ESTATE;
    const int n = (int)(P->ev_count < TIMING_SLOTS ? P->ev_count : TIMING_SLOTS);
    double total = 0.0;
    for (int i = 0; i < n; ++i) {
        const int slot = (int)((P->ev_count - 1 - i) % TIMING_SLOTS);
        CUDA_TRY(cudaEventSynchronize(P->ev1[slot]));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, P->ev0[slot], P->ev1[slot]));
        total += ms;
    }
    *count_out = n;
    *total_ms_out = total;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_dmma_peak(int iters, double* tflops_out, void* cuda_stream) {
    if (!tflops_out || iters < 1) return CHEB_DM_EINVAL;
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return CHEB_DM_ECUDA;
    CUDA_TRY(cudaGetDevice(&dev));
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* sink = nullptr;
    CUDA_TRY(cudaMalloc(&sink, sizeof(double) * 64));
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0));
    CUDA_TRY(cudaEventCreate(&e1));
    const int blocks = prop.multiProcessorCount * 2, threads = 512;
    dmma_peak_kernel<<<blocks, threads, 0, st>>>(iters / 8 + 1, sink);  // warm-up
    CUDA_TRY(cudaEventRecord(e0, st));
    dmma_peak_kernel<<<blocks, threads, 0, st>>>(iters, sink);
    CUDA_TRY(cudaEventRecord(e1, st));
    CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    const double flops = (double)blocks * (threads / 32) * (double)iters * DMMA_PEAK_CHAINS * 512.0;
    *tflops_out = flops / ((double)ms * 1e-3) * 1e-12;
    return CHEB_DM_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// cheb_dm_bounds_static (include/cheb_dm.h): Gershgorin bounds with the scratch in a fixed device array -- the one entry
// point that never allocates.  Everything it needs is in this block; no other code path uses it.
// ---------------------------------------------------------------------------------------------------------------------
// [0, 256): completion ticket (unsigned, must be zero when a call starts); then one (h_ii - R_i, h_ii + R_i) pair per row.
static __device__ __align__(256) unsigned char cheb_dm_static_scratch[256 + 16 * CHEB_DM_STATIC_MAX_N];

namespace {

constexpr int BS_THREADS = 256, BS_ROWS = BS_THREADS / 32;  // a warp per row

// `scratch` is the device address of cheb_dm_static_scratch, looked up by the host with cudaGetSymbolAddress.
__global__ void __launch_bounds__(BS_THREADS) bounds_static_kernel(const double* __restrict__ H, int N, long long ldh,
                                                                   unsigned char* __restrict__ scratch, double* __restrict__ out) {
    unsigned* ticket = reinterpret_cast<unsigned*>(scratch);
    double* rows = reinterpret_cast<double*>(scratch + 256);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int row = blockIdx.x * BS_ROWS + warp;
    if (row < N) {
        const double* hr = H + (long long)row * ldh;
        const bool vec = ((ldh & 1) == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
        double r = 0.0, hii = 0.0;
        if (vec) {
            const int jend = N & ~1;
            for (int j = 2 * lane; j < jend; j += 64) {
                const double2 v = __ldg(reinterpret_cast<const double2*>(hr + j));
                if (j == row) hii = v.x; else r += fabs(v.x);
                if (j + 1 == row) hii = v.y; else r += fabs(v.y);
            }
            if ((N & 1) && lane == 0) {
                const double v = hr[N - 1];
                if (N - 1 == row) hii = v; else r += fabs(v);
            }
        } else {
            for (int j = lane; j < N; j += 32) {
                const double v = hr[j];
                if (j == row) hii = v; else r += fabs(v);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            r += __shfl_xor_sync(0xffffffffu, r, o);
            hii += __shfl_xor_sync(0xffffffffu, hii, o);  // exactly one lane holds h_ii, the rest 0
        }
        if (lane == 0) {
            const bool fin = isfinite(r) && isfinite(hii);
            rows[2 * row] = fin ? hii - r : -INFINITY;
            rows[2 * row + 1] = fin ? hii + r : INFINITY;
        }
    }
    // the block that draws the last ticket reduces the rows of all blocks (min / max: the order does not matter)
    __shared__ unsigned s_last;
    __shared__ double s_lo[BS_ROWS], s_hi[BS_ROWS];
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1u) ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double lo = INFINITY, hi = -INFINITY;
    for (int i = threadIdx.x; i < N; i += BS_THREADS) {
        lo = fmin(lo, __ldcg(rows + 2 * i));
        hi = fmax(hi, __ldcg(rows + 2 * i + 1));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if (lane == 0) { s_lo[warp] = lo; s_hi[warp] = hi; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < BS_ROWS; ++q) { lo = fmin(lo, s_lo[q]); hi = fmax(hi, s_hi[q]); }
        if (lo == hi) { lo -= 1.0; hi += 1.0; }  // degenerate H = cI (reading A2-iv), as front_end_kernel
        out[0] = lo;
        out[1] = hi;
        *ticket = 0u;  // left at zero for the next call (the host clears it as well: an aborted call may not get here)
    }
}

// Device address of the scratch array, per device: cudaGetSymbolAddress once, with that device current.
constexpr int BS_MAX_DEVICES = 64;
unsigned char* g_static_scratch_ptr[BS_MAX_DEVICES];
int g_static_scratch_ok[BS_MAX_DEVICES];

}  // namespace

extern "C" cheb_dm_status_t cheb_dm_bounds_static(const double* dH, int N, long long ldh, double* d_bounds, void* cuda_stream) {
    if (!dH || !d_bounds || N < 1 || ldh < N) return CHEB_DM_EINVAL;
    if (N > CHEB_DM_STATIC_MAX_N) return CHEB_DM_ESIZE;
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= BS_MAX_DEVICES) return CHEB_DM_ECUDA;
    if (!__atomic_load_n(&g_static_scratch_ok[dev], __ATOMIC_ACQUIRE)) {
        // In host code the array's name is a host-side stand-in, not a device address: ask the runtime for the address on
        // the current device.  (Two threads racing here store the same value.)
        unsigned char* ptr = nullptr;
        if (cudaGetSymbolAddress((void**)&ptr, cheb_dm_static_scratch) != cudaSuccess || ptr == nullptr) {
            cudaGetLastError();
            return CHEB_DM_ECUDA;
        }
        g_static_scratch_ptr[dev] = ptr;
        __atomic_store_n(&g_static_scratch_ok[dev], 1, __ATOMIC_RELEASE);
    }
    unsigned char* scratch = g_static_scratch_ptr[dev];
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CUDA_TRY(cudaMemsetAsync(scratch, 0, 256, st));  // the ticket must start at zero whatever the last call left
    const int grid = (N + BS_ROWS - 1) / BS_ROWS;
    bounds_static_kernel<<<grid, BS_THREADS, 0, st>>>(dH, N, ldh, scratch, d_bounds);
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}
