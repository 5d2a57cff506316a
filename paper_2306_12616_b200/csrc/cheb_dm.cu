// cheb_dm.cu -- host side of the C ABI declared in include/cheb_dm.h: plan (block sizes, workspace,
// TMA descriptors, task/dependency tables) and the launches of the sm_100a kernels.  Product code;
// shares nothing with oracle/.  There is no CPU path: every step of the solve runs in the kernels of
// gemm_dmma.cuh / aux_kernels.cuh.
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
#include "giant_resident.cuh"

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
typedef GemmCfg<64, 64, 32, 16, 32, 6, 1> Cfg64x64w16;     //  8 consumer warps of 32x16, 192 KB ring, 1 CTA/SM
typedef GemmCfg<112, 64, 16, 32, 16, 6, 1> Cfg112x64;     // 14 consumer warps of 16x32, 132 KB ring, 1 CTA/SM (N ~ 1000: 144 tiles)

enum TileSel { TILE_AUTO = 0, TILE_128x128 = 1, TILE_128x64 = 2, TILE_64x64 = 3, TILE_64x32_W16 = 4, TILE_64x32_W32 = 5,
               TILE_128x64_W16 = 6, TILE_32x32 = 7, TILE_112x64 = 8, TILE_64x64_W16 = 9, TILE_LAST = 9 };

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

struct HostTaskMeta {
    int has_gemm;
};

}  // namespace

enum { TIMING_SLOTS = 256 };

struct cheb_dm_plan_s {
    int N, M, k, p, Nq;
    cheb_dm_options_t opt;
    int device, num_sms;
    int tile;  // TileSel actually used
    int BM, BN, BK, box_slabs;
    long long ld;        // padded leading dimension of workspace matrices (multiple of 16)
    size_t mat_elems;    // elements per workspace matrix
    int nmat;            // k + 2 (+ p when the sums are pre-formed)
    double* ws;          // nmat matrices
    // scalar tables (device)
    double *costab, *fn, *c, *gT, *dT, *Amat, *tau, *w, *dots, *one, *part;
    int front_grid;      // blocks of the cooperative front_end_kernel
    int preformed;       // 1: low-order sums G_l are formed by form_sums_kernel before the giant steps
    int sym;             // 1: symmetric-tile skipping in gemm_dmma_kernel
    int* sym_first;      // device: [tiles_n + 1] item prefix sums of a symmetric task
    int resident;        // 1: giant steps run in giant_resident_kernel (small N), baby steps in gemm_dmma_kernel
    int res_tiles_m, res_tiles_n, res_grid, res_smem;
    DevScalars* sc;
    CUtensorMap* maps;   // nmat descriptors
    int tma2d;
    // task tables
    int ntasks_solve;        // tasks [0, ntasks_solve) = the solve; [ntasks_solve, ntasks_all) = moments chain
    int ntasks_all;
    int nbaby;               // baby tasks are [0, nbaby)
    int product_task;        // index of the scratch task used by cheb_dm_product
    Task* tasks;             // device
    int* task_first;         // device, ntasks_all + 2
    std::vector<Task> h_tasks;
    std::vector<int> h_first;
    int* counters;           // device: [work counters | task_done | group_done | panel_done | error]
    size_t counters_ints;
    int off_work, off_task, off_group, off_panel, off_error;
    int panel_stride;
    int nwork;               // number of work counters (one per possible launch)
    // state
    int have_coeffs, explicit_bounds, have_moments, computed;
    double beta, mu, a, b;
    int last_launches;
    double flops_per_compute;
    size_t ws_bytes;
    // host-buffer entry point (cheb_dm_compute_host): device staging for H, D and tr D
    double *stage_H, *stage_D, *stage_tr;
    // pipelined host entry point (cheb_dm_compute_host_async): second staging slot, copy streams, events
    double *stage_H1, *stage_D1, *stage_tr1;
    cudaStream_t s_in, s_out;
    cudaEvent_t ev_in[2], ev_comp[2], ev_out[2];
    long long n_async;
    int pipe_ready;
    // optional per-tile timeline (cheb_dm_set_trace)
    TraceRec* trace_buf;
    int trace_on;
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

double* T_ptr(const cheb_dm_plan_s* P, int n) {  // T_n, 1 <= n <= k
    return P->ws + (size_t)(n - 1) * P->mat_elems;
}
int T_map(int n) { return n - 1; }
double* buf_ptr(const cheb_dm_plan_s* P, int i) { return P->ws + (size_t)(P->k + i) * P->mat_elems; }
int buf_map(const cheb_dm_plan_s* P, int i) { return P->k + i; }
double* G_ptr(const cheb_dm_plan_s* P, int l) { return P->ws + (size_t)(P->k + 2 + l) * P->mat_elems; }

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

}  // namespace

namespace {

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

void choose_tile(cheb_dm_plan_s* P) {
    int sel = P->opt.tile;
    if (sel < TILE_AUTO || sel > TILE_LAST) sel = TILE_AUTO;
    if (sel == TILE_AUTO) {
        // One product is the unit of the serial chain (giant steps), so pick the shape that minimises the time of
        // one product on this device: tiles per SM (whole waves, 1 CTA per SM) x tile area / main-loop efficiency.
        // Large N -> 128x128 (least L2 traffic per flop); N ~ 1000 -> 128x64; N ~ 500 -> 64x32 (128 tiles).
        // With symmetric-tile skipping only the lower-triangle tiles count (N <= 512: the giant steps run in the
        // resident kernel and the tile shape only serves the throughput-bound baby phase: full count, as measured).
        const int cand[5] = {TILE_128x128, TILE_128x64_W16, TILE_112x64, TILE_64x64_W16, TILE_64x32_W16};
        double best = 0.0;
        for (int c = 0; c < 5; ++c) {
            const TileShape t = tile_shape(cand[c]);
            const bool count_sym = P->sym && P->N > 32 * GR_MAX_KTILES;
            if (cand[c] == TILE_64x64_W16 && !count_sym) continue;
            const int tiles = count_sym ? sym_items(P->N, t.BM, t.BN) : ceil_div(P->N, t.BM) * ceil_div(P->N, t.BN);
            const double cost = (double)ceil_div(tiles, P->num_sms) * t.BM * t.BN / t.eff;
            if (sel == TILE_AUTO || cost < best) {
                sel = cand[c];
                best = cost;
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

Task blank_task(const cheb_dm_plan_s* P) {
    Task t;
    memset(&t, 0, sizeof(t));
    t.mapA = t.mapB = 0;
    t.ktiles = ceil_div(P->N, P->BK);
    t.tiles_m = ceil_div(P->N, P->BM);
    t.tiles_n = ceil_div(P->N, P->BN);
    t.sym = 0;
    t.nitems = t.tiles_m * t.tiles_n;
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

// Groups: 0 = baby steps of the solve, 1 = giant steps, 2 = moments chain, 3 = cheb_dm_product scratch.
enum { GROUP_BABY = 0, GROUP_GIANT = 1, GROUP_MOM = 2, GROUP_MISC = 3, NGROUPS = 4 };

void build_tasks(cheb_dm_plan_s* P) {
    const int k = P->k, p = P->p;
    std::vector<Task>& T = P->h_tasks;
    T.clear();
    const int tiles = ceil_div(P->N, P->BM) * ceil_div(P->N, P->BN);
    const int tiles_m = ceil_div(P->N, P->BM);
    // every matrix of the solve is a polynomial of X, hence symmetric: lower-triangle tiles only (option symmetric)
    const int stiles = P->sym ? sym_items(P->N, P->BM, P->BN) : tiles;

    // ---- baby steps: T_n = 2 T_l T_r - T_m (Eq. 7 / 22-23 / Algorithm 1) ----
    std::vector<BabyProd> sched = baby_schedule(k, P->opt.pairing);
    std::vector<int> task_of(k + 1, -1);  // task index that produces T_n (n >= 2)
    for (const BabyProd& bp : sched) {
        Task t = blank_task(P);
        t.mapA = T_map(bp.l);
        t.mapB = T_map(bp.r);
        t.group = GROUP_BABY;
        t.alpha = 2.0;
        if (bp.m == 0) {
            t.C = nullptr;
            t.diag_const = -1.0;  // - T_0 = -I
        } else {
            t.C = T_ptr(P, bp.m);
            t.ldc = P->ld;
            t.beta = -1.0;
        }
        t.Out = T_ptr(P, bp.n);
        t.ldo = P->ld;
        int deps[3] = {bp.l, bp.r, bp.m};
        for (int d = 0; d < 3; ++d) {
            const int n = deps[d];
            if (n < 2) continue;
            bool dup = false;
            for (int e = 0; e < d; ++e) dup = dup || (deps[e] == n);
            if (!dup) add_dep(t, DEP_TASK, task_of[n], stiles);
        }
        t.sym = P->sym;
        t.nitems = stiles;
        task_of[bp.n] = (int)T.size();
        T.push_back(t);
    }
    P->nbaby = (int)T.size();
    const int baby_tiles = P->nbaby * stiles;

    // ---- giant steps ----
    // CHEBYSHEV: B_l = G_l + 2 Y B_{l+1} - B_{l+2} (l = p-1..1), D = G_0 + Y B_1 - B_2, G_l = sum_i g_{i,l} T_i.
    // POWER    : acc_j = S_j + Y acc_{j+1} (Eq. 4), S_j = sum_i d_{i,j} T_i (Eq. 21).
    // B_l / acc_l lives in buf[l & 1]; Y = T_k.  Column panels of successive steps are independent chains, so
    // step l only waits for the SAME column panel of step l+1 (DEP_PANEL_N).
    const bool power = (P->opt.outer == CHEB_DM_OUTER_POWER);
    const double* coefT = power ? P->dT : P->gT;
    const int first_giant = (int)T.size();
    for (int l = p - 1; l >= 0; --l) {
        Task t = blank_task(P);
        t.group = GROUP_GIANT;
        const bool has_prod = (l + 1 <= p - 1);
        if (has_prod) {
            t.mapA = T_map(k);
            t.mapB = buf_map(P, (l + 1) & 1);
            t.alpha = (power || l == 0) ? 1.0 : 2.0;
            if (!power && l + 2 <= p - 1) {
                t.C = buf_ptr(P, (l + 2) & 1);
                t.ldc = P->ld;
                t.beta = -1.0;
            }
        } else {
            t.ktiles = 0;
        }
        if (l == 0) {
            t.out_is_user = 1;
        } else {
            t.Out = buf_ptr(P, l & 1);
            t.ldo = P->ld;
        }
        if (P->preformed) {
            // G_l / S_l was formed by form_sums_kernel (diagonal term included): one extra tile, weight 1
            t.sum_base = G_ptr(P, l);
            t.sum_count = 1;
            t.coef = P->one;
            t.diag_ptr = nullptr;
        } else {
            // low-order sum: T_1..T_{k-1} with coefficients row l of the table, T_0 = I through diag_ptr
            t.sum_base = T_ptr(P, 1);
            t.sum_count = k - 1;
            t.coef = coefT + (size_t)l * k + 1;
            t.diag_ptr = coefT + (size_t)l * k;
        }
        // early: the baby block (operands of the low-order sum); late: the same column panel of the previous step
        if (P->nbaby > 0) add_dep(t, DEP_GROUP, GROUP_BABY, baby_tiles);
        t.ndeps_early = t.ndeps;
        // (symmetric tiles: a panel also receives mirrored blocks from the tiles of other panels, so the step waits
        // for the whole previous step; the resident kernel keeps full tiles and panel chains)
        if (P->sym && !P->resident) {
            t.sym = 1;
            t.nitems = stiles;
            if (has_prod) add_dep(t, DEP_TASK, (int)T.size() - 1, stiles);
        } else if (has_prod) {
            add_dep(t, DEP_PANEL_N, (int)T.size() - 1, tiles_m);
        }
        T.push_back(t);
    }
    (void)first_giant;
    P->ntasks_solve = (int)T.size();

    // ---- moments chain (cheb_dm_moments): U_j = T_j(Y), U_{j+1} = 2 Y U_j - U_{j-1}, j = 1..p-2, with the
    // Frobenius products <U_{j+1}, T_i>, i < k, fused into the epilogue (dot_count).  U_j lives in buf[j & 1]
    // for j >= 2 (U_1 = Y = T_k, U_0 = I).
    for (int j = 1; j + 1 <= p - 1; ++j) {
        Task t = blank_task(P);
        t.group = GROUP_MOM;
        t.mapA = T_map(k);
        t.mapB = (j == 1) ? T_map(k) : buf_map(P, j & 1);
        t.alpha = 2.0;
        if (j == 1) {
            t.diag_const = -1.0;
        } else if (j == 2) {
            t.C = T_ptr(P, k);
            t.ldc = P->ld;
            t.beta = -1.0;
        } else {
            t.C = buf_ptr(P, (j - 1) & 1);
            t.ldc = P->ld;
            t.beta = -1.0;
        }
        t.Out = buf_ptr(P, (j + 1) & 1);
        t.ldo = P->ld;
        t.sum_base = T_ptr(P, 1);
        t.dot_count = k - 1;  // <U_{j+1}, T_i> for i = 1..k-1; slot k-1 = tr U_{j+1} (= <U, T_0>)
        t.dot_out = P->dots + (size_t)(j + 1) * tiles * k;  // slots of skipped tiles stay zero (memset at plan time)
        t.sym = P->sym;                                     // U_j = T_j(T_k) is symmetric too; dots weight mirrored blocks x2
        t.nitems = stiles;
        if (P->nbaby > 0) add_dep(t, DEP_GROUP, GROUP_BABY, baby_tiles);
        if (j >= 2) add_dep(t, DEP_TASK, (int)T.size() - 1, stiles);
        T.push_back(t);
    }
    P->ntasks_all = (int)T.size();

    // ---- scratch task of cheb_dm_product ----
    {
        Task t = blank_task(P);
        t.group = GROUP_MISC;
        t.mapA = buf_map(P, 0);
        t.mapB = buf_map(P, 1);
        t.out_is_user = 1;
        P->product_task = (int)T.size();
        T.push_back(t);
    }

    P->h_first.assign(T.size() + 1, 0);
    for (size_t i = 0; i < T.size(); ++i) P->h_first[i + 1] = P->h_first[i] + T[i].nitems;

    double nprod = 0;  // executed products, counting only the tiles that are computed
    const double res_frac = P->sym ? (double)(P->res_tiles_m + 1) / (2.0 * P->res_tiles_m) : 1.0;  // 32x32 lower-triangle tiles
    for (int i = 0; i < P->ntasks_solve; ++i) {
        if (T[i].ktiles <= 0) continue;
        nprod += (P->resident && i >= P->nbaby) ? res_frac : (double)T[i].nitems / (double)tiles;
    }
    P->flops_per_compute = nprod * 2.0 * (double)P->N * (double)P->N * (double)P->N;
}

cheb_dm_status_t encode_maps(cheb_dm_plan_s* P) {
    EncodeTiledFn enc = get_encode_fn();
    if (!enc) return CHEB_DM_ECUDA;
    const int nmaps = P->k + 2;  // operands of products: T_1..T_k and the two giant-step buffers
    std::vector<CUtensorMap> h(nmaps);
    const char* env2d = getenv("CHEB_DM_TMA2D");
    int want2d = (env2d && env2d[0] == '1') ? 1 : 0;
    for (int pass = 0; pass < 2; ++pass) {
        bool ok = true;
        for (int i = 0; i < nmaps && ok; ++i) {
            void* base = P->ws + (size_t)i * P->mat_elems;
            CUresult r;
            if (!want2d) {
                // {16 columns (128 B), N rows, ld/16 slabs}: a box of 4 slabs x BK rows lands in shared memory as
                // [slab][row][128 B] with the 128-byte swizzle keyed on the row.
                cuuint64_t dims[3] = {16, (cuuint64_t)P->N, (cuuint64_t)(P->ld / 16)};
                cuuint64_t strides[2] = {(cuuint64_t)P->ld * 8, 128};
                cuuint32_t box[3] = {16, (cuuint32_t)P->BK, (cuuint32_t)P->box_slabs};
                cuuint32_t estr[3] = {1, 1, 1};
                r = enc(&h[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base, dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            } else {
                cuuint64_t dims[2] = {(cuuint64_t)P->ld, (cuuint64_t)P->N};
                cuuint64_t strides[1] = {(cuuint64_t)P->ld * 8};
                cuuint32_t box[2] = {16, (cuuint32_t)P->BK};
                cuuint32_t estr[2] = {1, 1};
                r = enc(&h[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, base, dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            }
            ok = (r == CUDA_SUCCESS);
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

template <class Cfg, bool DOTS>
cheb_dm_status_t launch_inst(const LaunchArgs& la, int items, int num_sms, cudaStream_t st) {
    static bool attr_set = false;
    if (!attr_set) {
        CUDA_TRY(cudaFuncSetAttribute(gemm_dmma_kernel<Cfg, DOTS>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM_BYTES));
        attr_set = true;
    }
    int per_sm = 1;
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, gemm_dmma_kernel<Cfg, DOTS>, Cfg::THREADS, Cfg::SMEM_BYTES));
    if (per_sm < 1) return CHEB_DM_ECUDA;
    int grid = per_sm * num_sms;
    if (grid > items) grid = items;
    if (grid < 1) grid = 1;
    gemm_dmma_kernel<Cfg, DOTS><<<grid, Cfg::THREADS, Cfg::SMEM_BYTES, st>>>(la);
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}
template <class Cfg>
cheb_dm_status_t launch_cfg(const LaunchArgs& la, int items, int num_sms, cudaStream_t st, bool dots) {
    return dots ? launch_inst<Cfg, true>(la, items, num_sms, st) : launch_inst<Cfg, false>(la, items, num_sms, st);
}

// Launch tasks [t0, t1) as one persistent grid; `work_slot` selects the work counter.
cheb_dm_status_t launch_tasks(cheb_dm_plan_s* P, int t0, int t1, int use_deps, int work_slot, double* userD,
                              long long ldD, cudaStream_t st) {
    LaunchArgs la;
    la.tasks = P->tasks;
    la.task_first = P->task_first;
    la.maps = P->maps;
    la.work_counter = P->counters + P->off_work + work_slot;
    la.task_done = P->counters + P->off_task;
    la.panel_done = P->counters + P->off_panel;
    la.group_done = P->counters + P->off_group;
    la.panel_stride = P->panel_stride;
    la.task_begin = t0;
    la.task_end = t1;
    la.use_deps = use_deps;
    la.N = P->N;
    la.userD = userD;
    la.ldD = ldD;
    la.tma2d = P->tma2d;
    la.sym_first = P->sym_first;
    la.error_flag = P->counters + P->off_error;
    la.trace = P->trace_on ? P->trace_buf : nullptr;
    const int items = P->h_first[t1] - P->h_first[t0];
    ++P->last_launches;
    bool dots = false;  // the moments chain needs the instance whose epilogue forms the Frobenius products
    for (int t = t0; t < t1; ++t) dots = dots || (P->h_tasks[t].dot_out != nullptr);
    switch (P->tile) {
        case TILE_128x128: return launch_cfg<Cfg128x128>(la, items, P->num_sms, st, dots);
        case TILE_128x64: return launch_cfg<Cfg128x64>(la, items, P->num_sms, st, dots);
        case TILE_64x64: return launch_cfg<Cfg64x64>(la, items, P->num_sms, st, dots);
        case TILE_64x32_W16: return launch_cfg<Cfg64x32w16>(la, items, P->num_sms, st, dots);
        case TILE_64x32_W32: return launch_cfg<Cfg64x32w32>(la, items, P->num_sms, st, dots);
        case TILE_32x32: return launch_cfg<Cfg32x32>(la, items, P->num_sms, st, dots);
        case TILE_112x64: return launch_cfg<Cfg112x64>(la, items, P->num_sms, st, dots);
        case TILE_64x64_W16: return launch_cfg<Cfg64x64w16>(la, items, P->num_sms, st, dots);
        default: return launch_cfg<Cfg128x64w16>(la, items, P->num_sms, st, dots);
    }
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
        case CHEB_DM_EUNSUPPORTED: return "unsupported dtype";
        case CHEB_DM_ENOCONV: return "power-basis outer recursion would lose accuracy (use the Chebyshev outer recursion)";
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
    cudaFree(P->dots);
    cudaFree(P->one);
    cudaFree(P->part);
    cudaFree(P->sym_first);
    cudaFree(P->sc);
    cudaFree(P->maps);
    cudaFree(P->tasks);
    cudaFree(P->task_first);
    cudaFree(P->counters);
    cudaFree(P->stage_H);
    cudaFree(P->stage_D);
    cudaFree(P->stage_tr);
    cudaFree(P->stage_H1);
    cudaFree(P->stage_D1);
    cudaFree(P->stage_tr1);
    if (P->pipe_ready) {
        cudaStreamDestroy(P->s_in);
        cudaStreamDestroy(P->s_out);
        for (int i = 0; i < 2; ++i) {
            cudaEventDestroy(P->ev_in[i]);
            cudaEventDestroy(P->ev_comp[i]);
            cudaEventDestroy(P->ev_out[i]);
        }
    }
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
    if (o.pairing != CHEB_DM_PAIR_ALG1 && o.pairing != CHEB_DM_PAIR_SERIAL && o.pairing != CHEB_DM_PAIR_BALANCED) return CHEB_DM_EINVAL;
    if (o.fuse_sums < 0 || o.fuse_sums > 2) return CHEB_DM_EINVAL;
    if (o.giant < 0 || o.giant > 2) return CHEB_DM_EINVAL;
    if (o.symmetric < 0 || o.symmetric > 2) return CHEB_DM_EINVAL;
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
    P->opt = o; P->opt.k = k; P->opt.p = p;
    P->device = dev; P->num_sms = prop.multiProcessorCount;
    int nq = 1;
    while (nq < 4 * M_terms) nq <<= 1;  // N_q = 2^ceil(log2(4M)) (cheb_dm.h)
    P->Nq = nq;
    P->sym = (o.symmetric != 1) ? 1 : 0;
    P->opt.symmetric = P->sym ? 2 : 1;
    P->sym_first = nullptr;
    choose_tile(P);
    P->ld = ((long long)N + 15) / 16 * 16;
    P->mat_elems = (((size_t)N * (size_t)P->ld) + 127) / 128 * 128;
    // Giant steps in the resident-multiplier kernel: N <= 512 (32 rows of T_k fit in shared memory), operand maps
    // with BK = 32 and 2-slab boxes (the 64x32 / 32x32 tile shapes), grouped scheduling, at least one product.
    P->resident = 0;
    P->res_tiles_m = P->res_tiles_n = ceil_div(N, 32);
    P->res_grid = P->sym ? (P->res_tiles_m * (P->res_tiles_m + 1)) / 2 : P->res_tiles_m * ceil_div(P->res_tiles_n, 2);
    P->res_smem = giant_resident_smem_bytes(ceil_div(N, GR_BK));
    if (o.giant != 1 && N <= 32 * GR_MAX_KTILES && p >= 2 && P->BK == GR_BK && P->box_slabs == 2 &&
        o.sched == CHEB_DM_SCHED_GROUPED && P->res_grid <= P->num_sms) {
        if (cudaFuncSetAttribute(giant_resident_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, P->res_smem) == cudaSuccess) {
            int per_sm = 0;
            if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, giant_resident_kernel, GR_THREADS, P->res_smem) == cudaSuccess && per_sm >= 1)
                P->resident = 1;
        }
        cudaGetLastError();
    }
    P->opt.giant = P->resident ? 2 : 1;
    // a-5: fused (epilogue reads T_1..T_{k-1}: p (k-1) mat bytes per solve) while the baby block stays L2-resident,
    // pre-formed (form_sums_kernel: (ceil(p/16) (k-1) + p) mat bytes) once it does not.
    {
        int mode = o.fuse_sums;
        if (mode == 0) mode = ((double)k * (double)P->mat_elems * 8.0 > 96.0 * 1024 * 1024 && k > 2 && p > 1) ? 2 : 1;
        P->preformed = (mode == 2) ? 1 : 0;
        P->opt.fuse_sums = mode;
    }
    if (P->resident) {  // the resident kernel forms the sums itself (each CTA its own tiles) and parks them in G_l
        P->preformed = 1;
        P->opt.fuse_sums = 2;
    }
    P->nmat = k + 2 + (P->preformed ? p : 0);
    P->ws = nullptr; P->costab = P->fn = P->c = P->gT = P->dT = P->Amat = P->tau = P->w = P->dots = P->one = P->part = nullptr;
    P->sc = nullptr; P->maps = nullptr; P->tasks = nullptr; P->task_first = nullptr; P->counters = nullptr;
    P->have_coeffs = P->explicit_bounds = P->have_moments = P->computed = 0;
    P->last_launches = 0;
    P->stage_H = P->stage_D = P->stage_tr = nullptr;
    P->stage_H1 = P->stage_D1 = P->stage_tr1 = nullptr;
    P->pipe_ready = 0;
    P->n_async = 0;
    P->timing = 0; P->ev_count = 0;
    P->trace_buf = nullptr; P->trace_on = 0;
    for (int i = 0; i < TIMING_SLOTS; ++i) P->ev0[i] = P->ev1[i] = nullptr;

    const int tiles = ceil_div(N, P->BM) * ceil_div(N, P->BN);
    const size_t kp = (size_t)k * p;
    P->ws_bytes = sizeof(double) * P->mat_elems * P->nmat;
    bool ok = true;
    ok = ok && cudaMalloc(&P->ws, P->ws_bytes) == cudaSuccess;
    ok = ok && cudaMalloc(&P->costab, sizeof(double) * 4 * nq) == cudaSuccess;
    ok = ok && cudaMalloc(&P->fn, sizeof(double) * nq) == cudaSuccess;
    ok = ok && cudaMalloc(&P->c, sizeof(double) * kp) == cudaSuccess;
    ok = ok && cudaMalloc(&P->gT, sizeof(double) * kp) == cudaSuccess;
    ok = ok && cudaMalloc(&P->dT, sizeof(double) * kp) == cudaSuccess;
    ok = ok && cudaMalloc(&P->Amat, sizeof(double) * p * p) == cudaSuccess;
    ok = ok && cudaMalloc(&P->tau, sizeof(double) * kp) == cudaSuccess;
    ok = ok && cudaMalloc(&P->w, sizeof(double) * nq) == cudaSuccess;
    ok = ok && cudaMalloc(&P->dots, sizeof(double) * ((size_t)(p + 1) * tiles * k + (size_t)2 * k * 16)) == cudaSuccess;
    ok = ok && cudaMalloc(&P->sc, sizeof(DevScalars)) == cudaSuccess;
    ok = ok && cudaMalloc(&P->one, sizeof(double)) == cudaSuccess;
    {
        int per_sm = 0;
        ok = ok && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, front_end_kernel, 512, 0) == cudaSuccess && per_sm >= 1;
        int want = ceil_div(N, 16);
        if (ceil_div((int)kp, 16) > want) want = ceil_div((int)kp, 16);
        if (ceil_div(nq, 512) > want) want = ceil_div(nq, 512);
        P->front_grid = want < P->num_sms ? want : P->num_sms;
        ok = ok && cudaMalloc(&P->part, sizeof(double) * 2 * P->num_sms) == cudaSuccess;
    }
    ok = ok && cudaMalloc(&P->maps, sizeof(CUtensorMap) * P->nmat) == cudaSuccess;
    ok = ok && cudaMalloc(&P->stage_H, sizeof(double) * (size_t)N * N) == cudaSuccess;
    ok = ok && cudaMalloc(&P->stage_D, sizeof(double) * (size_t)N * N) == cudaSuccess;
    ok = ok && cudaMalloc(&P->stage_tr, sizeof(double)) == cudaSuccess;
    for (int i = 0; i < TIMING_SLOTS && ok; ++i)
        ok = cudaEventCreate(&P->ev0[i]) == cudaSuccess && cudaEventCreate(&P->ev1[i]) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        cheb_dm_destroy(P);
        return CHEB_DM_EALLOC;
    }
    P->ws_bytes += sizeof(double) * (2 * (size_t)N * N + 4 * (size_t)nq + 2 * nq + 4 * kp + (size_t)p * p + (size_t)(p + 1) * tiles * k);

    cheb_dm_status_t st = CHEB_DM_OK;
    do {
        if (cudaMemset(P->ws, 0, sizeof(double) * P->mat_elems * P->nmat) != cudaSuccess) { st = CHEB_DM_ECUDA; break; }
        cudaMemset(P->dots, 0, sizeof(double) * ((size_t)(p + 1) * tiles * k + (size_t)2 * k * 16));
        cudaMemset(P->dT, 0, sizeof(double) * kp);
        cudaMemset(P->gT, 0, sizeof(double) * kp);
        cudaMemset(P->c, 0, sizeof(double) * kp);
        cudaMemset(P->sc, 0, sizeof(DevScalars));
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
            std::vector<int> pf(tn_ + 1, 0);
            for (int tn = 0; tn < tn_; ++tn) {
                const int tm0 = sym_tm0(tn, P->BM, P->BN);
                pf[tn + 1] = pf[tn] + (tm0 < tm_ ? tm_ - tm0 : 0);
            }
            if (cudaMalloc(&P->sym_first, sizeof(int) * pf.size()) != cudaSuccess) { cudaGetLastError(); st = CHEB_DM_EALLOC; break; }
            if (cudaMemcpy(P->sym_first, pf.data(), sizeof(int) * pf.size(), cudaMemcpyHostToDevice) != cudaSuccess) { st = CHEB_DM_ECUDA; break; }
        }
        st = encode_maps(P);
        if (st != CHEB_DM_OK) break;
        build_tasks(P);
        const int nt = (int)P->h_tasks.size();
        P->panel_stride = ceil_div(N, 16);  // >= the number of column panels of every kernel (narrowest panel: 16)
        P->nwork = nt + 4;
        P->off_work = 0;
        P->off_task = P->off_work + P->nwork;
        P->off_group = P->off_task + nt;
        P->off_error = P->off_group + NGROUPS;
        P->off_panel = P->off_error + 1;
        P->counters_ints = (size_t)P->off_panel + (size_t)nt * P->panel_stride;
        if (cudaMalloc(&P->tasks, sizeof(Task) * nt) != cudaSuccess ||
            cudaMalloc(&P->task_first, sizeof(int) * (nt + 1)) != cudaSuccess ||
            cudaMalloc(&P->counters, sizeof(int) * P->counters_ints) != cudaSuccess) {
            cudaGetLastError();
            st = CHEB_DM_EALLOC;
            break;
        }
        if (cudaMemcpy(P->tasks, P->h_tasks.data(), sizeof(Task) * nt, cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemcpy(P->task_first, P->h_first.data(), sizeof(int) * (nt + 1), cudaMemcpyHostToDevice) != cudaSuccess ||
            cudaMemset(P->counters, 0, sizeof(int) * P->counters_ints) != cudaSuccess) {
            st = CHEB_DM_ECUDA;
            break;
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

}  // extern "C"

namespace {

// Steps a-1 .. a-3 on the stream, one cooperative launch: counters reset, bounds (+ rescale of H into T_1), c_n,
// g (and d).
cheb_dm_status_t front_end(cheb_dm_plan_s* P, const double* dH, cudaStream_t st) {
    FrontArgs fa;
    fa.H = dH;
    fa.N = P->N;
    fa.X = T_ptr(P, 1);
    fa.ldx = P->ld;
    fa.sc = P->sc;
    fa.explicit_bounds = P->explicit_bounds;
    fa.a = P->a;
    fa.b = P->b;
    fa.part = P->part;
    fa.counters = P->counters;
    fa.ncounters = (int)P->counters_ints;
    fa.beta = P->beta;
    fa.mu = P->mu;
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
    CUDA_TRY(cudaLaunchCooperativeKernel((const void*)front_end_kernel, dim3(P->front_grid), dim3(512), args, 0, st));
    ++P->last_launches;
    return CHEB_DM_OK;
}

cheb_dm_status_t run_tasks(cheb_dm_plan_s* P, int t0, int t1, double* userD, long long ldD, cudaStream_t st) {
    if (t1 <= t0) return CHEB_DM_OK;
    if (P->opt.sched == CHEB_DM_SCHED_GROUPED) return launch_tasks(P, t0, t1, 1, t0, userD, ldD, st);
    for (int t = t0; t < t1; ++t) {
        cheb_dm_status_t s = launch_tasks(P, t, t + 1, 0, t, userD, ldD, st);
        if (s != CHEB_DM_OK) return s;
    }
    return CHEB_DM_OK;
}

// Giant steps of the solve (tasks [nbaby, ntasks_solve)) in the resident-multiplier kernel; cooperative launch
// because its CTAs wait on one another's panel counters.
cheb_dm_status_t run_giant_resident(cheb_dm_plan_s* P, double* userD, long long ldD, cudaStream_t st) {
    GiantArgs ga;
    ga.tasks = P->tasks;
    ga.maps = P->maps;
    ga.first_task = P->nbaby;
    ga.nsteps = P->ntasks_solve - P->nbaby;
    ga.N = P->N;
    ga.ktiles = ceil_div(P->N, GR_BK);
    ga.tiles_m = P->res_tiles_m;
    ga.tiles_n = P->res_tiles_n;
    ga.panel_done = P->counters + P->off_panel;
    ga.panel_stride = P->panel_stride;
    ga.userD = userD;
    ga.ldD = ldD;
    ga.tma2d = P->tma2d;
    ga.error_flag = P->counters + P->off_error;
    ga.trace = P->trace_on ? P->trace_buf : nullptr;
    ga.trace_base = P->h_first.back();
    ga.coefT = (P->opt.outer == CHEB_DM_OUTER_POWER) ? P->dT : P->gT;
    ga.Tbase = T_ptr(P, 1);
    ga.Gbase = G_ptr(P, 0);
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

bool device_ok(const cheb_dm_plan_s* P) {
    int dev = -1;
    return cudaGetDevice(&dev) == cudaSuccess && dev == P->device;
}

}  // namespace

extern "C" {

cheb_dm_status_t cheb_dm_compute(cheb_dm_plan_t P, const double* dH, double* dD, void* cuda_stream) {
    if (!P || !dH || !dD || dH == dD) return CHEB_DM_EINVAL;
    if (!P->have_coeffs) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    P->last_launches = 0;
    cheb_dm_status_t s = front_end(P, dH, st);  // also zeroes the scheduler counters
    if (s != CHEB_DM_OK) return s;
    const int slot = (int)(P->ev_count % TIMING_SLOTS);
    if (P->timing) CUDA_TRY(cudaEventRecord(P->ev0[slot], st));
    if (P->resident) {
        s = run_tasks(P, 0, P->nbaby, dD, P->N, st);
        if (s != CHEB_DM_OK) return s;
        s = run_giant_resident(P, dD, P->N, st);
    } else if (P->preformed) {
        s = run_tasks(P, 0, P->nbaby, dD, P->N, st);
        if (s != CHEB_DM_OK) return s;
        const double* coefT = (P->opt.outer == CHEB_DM_OUTER_POWER) ? P->dT : P->gT;
        const char* scalar_sums = getenv("CHEB_DM_SCALAR_SUMS");
        if (scalar_sums && scalar_sums[0] == '1') {  // FP64-FMA version (ablation)
            const long long pairs = (long long)P->N * P->ld / 2;
            dim3 grid((unsigned)((pairs + 255) / 256), (unsigned)ceil_div(P->p, SUMS_CHUNK));
            form_sums_kernel<<<grid, 256, sizeof(double) * P->k * SUMS_CHUNK, st>>>(T_ptr(P, 1), (long long)P->mat_elems, P->ld, P->N, P->k,
                                                                                  P->p, coefT, G_ptr(P, 0), P->sym ? P->BM : 0, P->BN);
        } else {
            const long long warps = ((long long)P->N * P->ld + 31) / 32;
            dim3 grid((unsigned)((warps + 7) / 8), (unsigned)ceil_div(P->p, SUMS_CHUNK));
            const size_t smem = sizeof(double) * (size_t)((((P->k - 1) + 3) & ~3) + 1) * SUMS_CHUNK;
            form_sums_dmma_kernel<<<grid, 256, smem, st>>>(T_ptr(P, 1), (long long)P->mat_elems, P->ld, P->N, P->k, P->p, coefT,
                                                           G_ptr(P, 0), P->sym ? P->BM : 0, P->BN);
        }
        ++P->last_launches;
        CUDA_TRY(cudaGetLastError());
        s = run_tasks(P, P->nbaby, P->ntasks_solve, dD, P->N, st);
    } else {
        s = run_tasks(P, 0, P->ntasks_solve, dD, P->N, st);
    }
    if (s != CHEB_DM_OK) return s;
    if (P->timing) {
        CUDA_TRY(cudaEventRecord(P->ev1[slot], st));
        ++P->ev_count;
    }
    P->computed = 1;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_compute_host(cheb_dm_plan_t P, const double* hH, double* hD, double* h_trace, void* cuda_stream) {
    if (!P || !hH || !hD || hH == hD) return CHEB_DM_EINVAL;
    if (!P->have_coeffs) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bytes = sizeof(double) * (size_t)P->N * P->N;
    CUDA_TRY(cudaMemcpyAsync(P->stage_H, hH, bytes, cudaMemcpyHostToDevice, st));
    cheb_dm_status_t s = cheb_dm_compute(P, P->stage_H, P->stage_D, cuda_stream);
    if (s != CHEB_DM_OK) return s;
    if (h_trace) {
        trace_kernel<<<1, 1024, 0, st>>>(P->stage_D, P->N, P->N, P->stage_tr);
        ++P->last_launches;
        CUDA_TRY(cudaGetLastError());
        CUDA_TRY(cudaMemcpyAsync(h_trace, P->stage_tr, sizeof(double), cudaMemcpyDeviceToHost, st));
    }
    CUDA_TRY(cudaMemcpyAsync(hD, P->stage_D, bytes, cudaMemcpyDeviceToHost, st));
    return cheb_dm_check(P, cuda_stream);  // synchronises the stream
}

cheb_dm_status_t cheb_dm_compute_host_async(cheb_dm_plan_t P, const double* hH, double* hD, double* h_trace, void* cuda_stream) {
    if (!P || !hH || !hD || hH == hD) return CHEB_DM_EINVAL;
    if (!P->have_coeffs) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t bytes = sizeof(double) * (size_t)P->N * P->N;
    if (!P->pipe_ready) {
        bool ok = cudaMalloc(&P->stage_H1, bytes) == cudaSuccess && cudaMalloc(&P->stage_D1, bytes) == cudaSuccess &&
                  cudaMalloc(&P->stage_tr1, sizeof(double)) == cudaSuccess;
        if (!ok) { cudaGetLastError(); return CHEB_DM_EALLOC; }
        CUDA_TRY(cudaStreamCreateWithFlags(&P->s_in, cudaStreamNonBlocking));
        CUDA_TRY(cudaStreamCreateWithFlags(&P->s_out, cudaStreamNonBlocking));
        for (int i = 0; i < 2; ++i) {
            CUDA_TRY(cudaEventCreateWithFlags(&P->ev_in[i], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&P->ev_comp[i], cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&P->ev_out[i], cudaEventDisableTiming));
        }
        P->pipe_ready = 1;
    }
    const int slot = (int)(P->n_async & 1);
    double* sH = slot ? P->stage_H1 : P->stage_H;
    double* sD = slot ? P->stage_D1 : P->stage_D;
    double* sT = slot ? P->stage_tr1 : P->stage_tr;
    // H2D of this call: the slot's previous occupant (call n-2) must have been consumed by its kernels
    if (P->n_async >= 2) CUDA_TRY(cudaStreamWaitEvent(P->s_in, P->ev_comp[slot], 0));
    CUDA_TRY(cudaMemcpyAsync(sH, hH, bytes, cudaMemcpyHostToDevice, P->s_in));
    CUDA_TRY(cudaEventRecord(P->ev_in[slot], P->s_in));
    // kernels, in call order on the caller's stream: need this call's H and the slot's D / tr copied out (call n-2)
    CUDA_TRY(cudaStreamWaitEvent(st, P->ev_in[slot], 0));
    if (P->n_async >= 2) CUDA_TRY(cudaStreamWaitEvent(st, P->ev_out[slot], 0));
    cheb_dm_status_t s = cheb_dm_compute(P, sH, sD, cuda_stream);
    if (s != CHEB_DM_OK) return s;
    if (h_trace) {
        trace_kernel<<<1, 1024, 0, st>>>(sD, P->N, P->N, sT);
        ++P->last_launches;
        CUDA_TRY(cudaGetLastError());
    }
    CUDA_TRY(cudaEventRecord(P->ev_comp[slot], st));
    // D2H of this call
    CUDA_TRY(cudaStreamWaitEvent(P->s_out, P->ev_comp[slot], 0));
    if (h_trace) CUDA_TRY(cudaMemcpyAsync(h_trace, sT, sizeof(double), cudaMemcpyDeviceToHost, P->s_out));
    CUDA_TRY(cudaMemcpyAsync(hD, sD, bytes, cudaMemcpyDeviceToHost, P->s_out));
    CUDA_TRY(cudaEventRecord(P->ev_out[slot], P->s_out));
    ++P->n_async;
    return CHEB_DM_OK;
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
    DevScalars h;
    CUDA_TRY(cudaMemcpyAsync(&flag, P->counters + P->off_error, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaMemcpyAsync(&h, P->sc, sizeof(h), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    CUDA_TRY(cudaGetLastError());
    if (flag) return CHEB_DM_ECUDA;
    if (h.bad_bounds) return CHEB_DM_EBOUNDS;
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_set_trace(cheb_dm_plan_t P, int enable) {
    if (!P) return CHEB_DM_EINVAL;
    if (enable && !P->trace_buf) {
        const size_t n = (size_t)P->h_first.back() + (size_t)P->p * P->res_tiles_m * P->res_tiles_n;
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
    int n = P->h_first[P->resident ? P->nbaby : P->ntasks_solve];  // items of one solve (generic kernel)
    if (n > max_records) n = max_records;
    CUDA_TRY(cudaDeviceSynchronize());
    CUDA_TRY(cudaMemcpy(out, P->trace_buf, sizeof(TraceRec) * (size_t)n, cudaMemcpyDeviceToHost));
    if (P->resident) {  // followed by the tiles of the resident giant-step kernel
        int m = P->p * P->res_tiles_m * P->res_tiles_n;
        std::vector<TraceRec> tmp((size_t)m);
        CUDA_TRY(cudaMemcpy(tmp.data(), P->trace_buf + P->h_first.back(), sizeof(TraceRec) * (size_t)m, cudaMemcpyDeviceToHost));
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

cheb_dm_status_t cheb_dm_trace(cheb_dm_plan_t P, const double* dD, double* trace_out, void* cuda_stream) {
    if (!P || !dD || !trace_out) return CHEB_DM_EINVAL;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    trace_kernel<<<1, 1024, 0, st>>>(dD, P->N, P->N, trace_out);
    CUDA_TRY(cudaGetLastError());
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_get_bounds(cheb_dm_plan_t P, double* bounds_out, void* cuda_stream) {
    if (!P || !bounds_out) return CHEB_DM_EINVAL;
    if (!P->computed) return CHEB_DM_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    DevScalars h;
    CUDA_TRY(cudaMemcpyAsync(&h, P->sc, sizeof(h), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (h.bad_bounds || !isfinite(h.a) || !isfinite(h.b)) return CHEB_DM_EBOUNDS;
    bounds_out[0] = h.a;
    bounds_out[1] = h.b;
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
    unpad_copy_kernel<<<P->num_sms * 4, 256, 0, st>>>(T_ptr(P, n), P->ld, P->N, dOut);
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
    pad_copy_kernel<<<P->num_sms * 4, 256, 0, st>>>(dA, P->N, buf_ptr(P, 0), P->ld);
    pad_copy_kernel<<<P->num_sms * 4, 256, 0, st>>>(dB, P->N, buf_ptr(P, 1), P->ld);
    Task t = P->h_tasks[P->product_task];
    t.alpha = alpha;
    t.beta = beta;
    t.C = dC;
    t.ldc = P->N;
    CUDA_TRY(cudaMemcpyAsync(P->tasks + P->product_task, &t, sizeof(Task), cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemsetAsync(P->counters + P->off_work + P->product_task, 0, sizeof(int), st));
    const int save = P->last_launches;
    cheb_dm_status_t s = launch_tasks(P, P->product_task, P->product_task + 1, 0, P->product_task, dOut, P->N, st);
    P->last_launches = save;
    // the pageable-source copy above is staged by the runtime before it returns, so `t` may go out of scope
    return s;
}

}  // extern "C"

extern "C" {

cheb_dm_status_t cheb_dm_moments(cheb_dm_plan_t P, const double* dH, double* tau_host, void* cuda_stream) {
    if (!P || !dH) return CHEB_DM_EINVAL;
    if (!P->have_coeffs) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int k = P->k, p = P->p;
    const int tiles = ceil_div(P->N, P->BM) * ceil_div(P->N, P->BN);
    P->last_launches = 0;
    cheb_dm_status_t s = front_end(P, dH, st);  // counters reset, bounds + rescale (its coefficient tables are not used here)
    if (s != CHEB_DM_OK) return s;
    s = run_tasks(P, 0, P->nbaby, nullptr, 0, st);
    if (s != CHEB_DM_OK) return s;
    // j = 1: U_1 = T_k is a baby-step output, its products with T_1..T_{k-1} and all tr T_n come from one pass
    const int nchunks = 16;
    double* part1 = P->dots + (size_t)(p + 1) * tiles * k;  // (k-1) + 1 + k rows of nchunks partials
    {
        dim3 grid(2 * k, nchunks);
        frob_partial_kernel<<<grid, 256, 0, st>>>(T_ptr(P, k), T_ptr(P, 1), (long long)P->mat_elems, P->ld, P->N, k - 1, k, part1);
        ++P->last_launches;
    }
    // the chain tasks reuse group/task counters; the baby group counter is already complete
    if (P->ntasks_all > P->ntasks_solve) {
        if (P->opt.sched == CHEB_DM_SCHED_GROUPED)
            s = launch_tasks(P, P->ntasks_solve, P->ntasks_all, 1, P->ntasks_solve, nullptr, 0, st);
        else
            s = run_tasks(P, P->ntasks_solve, P->ntasks_all, nullptr, 0, st);
        if (s != CHEB_DM_OK) return s;
    }
    moments_kernel<<<1, 256, 0, st>>>(part1, nchunks, P->dots, tiles, k, p, P->N, P->tau);
    ++P->last_launches;
    CUDA_TRY(cudaGetLastError());
    P->have_moments = 1;
    P->computed = 1;
    if (tau_host) {
        CUDA_TRY(cudaMemcpyAsync(tau_host, P->tau, sizeof(double) * (size_t)k * p, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(cudaStreamSynchronize(st));
    }
    return CHEB_DM_OK;
}

cheb_dm_status_t cheb_dm_solve_mu(cheb_dm_plan_t P, double beta, double n_occ, int iters, double* mu_out,
                                  void* cuda_stream) {
    if (!P || !mu_out || iters < 1 || !isfinite(beta) || !(beta > 0.0) || !isfinite(n_occ)) return CHEB_DM_EINVAL;
    if (!P->have_moments) return CHEB_DM_ESTATE;
    if (!device_ok(P)) return CHEB_DM_ECUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    mu_weights_kernel<<<P->Nq, 128, 0, st>>>(P->tau, P->costab, P->Nq, P->M, P->w);
    mu_bisect_kernel<<<1, 1024, 0, st>>>(P->sc, beta, n_occ, iters, P->costab, P->Nq, P->w);
    CUDA_TRY(cudaGetLastError());
    DevScalars h;
    CUDA_TRY(cudaMemcpyAsync(&h, P->sc, sizeof(h), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (h.bad_bounds) return CHEB_DM_EBOUNDS;
    *mu_out = h.mu;
    return CHEB_DM_OK;
}

}  // extern "C"
