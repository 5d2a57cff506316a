// ozaki.cuh -- FP64-accurate product of two symmetric matrices on the Blackwell tensor path proper
// (SURVEY 8(f)-4): error-free slicing of the FP64 operands into int8 digits, the digit products on
// tcgen05.mma kind::i8 (SASS UTCIMMA) with int32 accumulators in tensor memory, recombination in FP64.
// sm_100a has no tcgen05 kind::f64 (the products of the solve run on DMMA.8x8x4, gemm_dmma.cuh); this is the
// only route past the DMMA issue rate for the products  T_{a+b} = 2 T_a T_b - T_|a-b|  (Eq. 7) and
// the Horner steps of Eq. (4).  Used by the stand-alone product cheb_dm_product_sliced and, with the plan
// option sliced_solve, for every product of cheb_dm_compute (one launch per product + one slicing pass per result).
// Product code; shares nothing with oracle/.
//
// Slicing (per row i of a symmetric operand; the row of B^T = B is the column of B):
//     a_ik = 2^{e_i} ( sum_{s<S} q_s[i][k] 2^{-6-7s} + rho ),   q_s in [-64, 64] (int8),  |rho| <= 2^{-7S},
// with 2^{e_i} > max_k |a_ik|:  t_0 = a 2^{6-e},  q_s = rint(t_s),  t_{s+1} = (t_s - q_s) 2^7  -- every step exact.
// Product:  (A B)_ij = 2^{e_i+f_j-12} sum_{d} 2^{-7d} P_d[i][j] + O(K 2^{e_i+f_j-7S}),
//     P_d = sum_{s+t=d} sum_k q^A_s[i][k] q^B_t[j][k]      exactly in int32:  |P_d| <= (d+1) K 64^2 < 2^31 for K <= 65535,
// keeping d < S (the dropped digit products are below the slicing error).  S(S+1)/2 int8 products: 36 for S = 8,
// for which the error bound K (S+1) 2^{-7S} 2^{e_i+f_j} is below the rounding error of an FP64 dot product.
//
// Kernel: one CTA per 128 x 64 output tile (persistent, static tile order), cta_group::1.  ALL S accumulators
// P_0..P_{S-1} live in tensor memory at once (S x 64 columns <= 512), so every digit tile is fetched once per k-block
// and used by up to S MMAs: S(S+1)/2 MMA blocks per 2S tile loads (a plain int8 GEMM loads 2 per block and is
// L2-bound on this part).  k-block = 64 int8 (64-byte swizzle rows), stage = S A-tiles (128 x 64 B) + S B-tiles
// (64 x 64 B), two stages.  Warp 0: TMA producer, warp 1: MMA issuer (one lane), warp 2: TMEM allocator, warps 4-11:
// epilogue (tcgen05.ld of the S accumulators, Horner recombination in FP64, scaling, alpha/beta, store).
#pragma once
#include "common.cuh"

namespace chebdm {

constexpr int OZ_MAX_S = 8;
constexpr int OZ_BM = 128, OZ_BN = 64, OZ_BK = 64;          // output tile, k-block in int8 elements (= bytes)
constexpr int OZ_A_TILE = OZ_BM * OZ_BK, OZ_B_TILE = OZ_BN * OZ_BK;   // 8 KB, 4 KB
constexpr int OZ_STAGES = 2;
constexpr int OZ_THREADS = 384;                               // warps 0-3: TMA, MMA issue, TMEM allocation, idle; warps 4-11: epilogue
constexpr int OZ_BAND = 16;                                  // column tiles per raster band (L2 reuse of the digit strips)

// ---- tcgen05 wrappers ----
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_alloc512(uint32_t smem_slot) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_slot) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tc_dealloc512(uint32_t taddr) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(taddr) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, int8 x int8 -> int32, M = 128, N = 64, K = 32 per instruction
__device__ __forceinline__ void tc_mma_i8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// arrive on an mbarrier when every MMA issued so far by this thread has completed (implies fence::before_thread_sync)
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tc_ld8(uint32_t taddr, int (&v)[8]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor, K-major operand tile of 64-byte rows with the 64-byte swizzle: 8-row groups are
// 512 bytes apart (stride byte offset), the leading byte offset is unused for swizzled K-major tiles, descriptor
// version 1 (sm_100), layout type 4 = SWIZZLE_64B.  Advancing by one K = 32 instruction adds 32 bytes to the start.
__device__ __forceinline__ uint64_t oz_smem_desc(uint32_t saddr) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr & 0x3FFFFu) >> 4);      // [0,14)  start address >> 4
    d |= (uint64_t)1 << 16;                         // [16,30) leading byte offset >> 4 (ignored)
    d |= (uint64_t)(512 >> 4) << 32;                // [32,46) stride byte offset >> 4
    d |= (uint64_t)1 << 46;                         // [46,48) descriptor version
    d |= (uint64_t)4 << 61;                         // [61,64) swizzle mode: 64 B
    return d;
}
// Instruction descriptor of kind::i8: D = S32 (2 at [4,6)), A and B signed int8 (1 at [7,10), [10,13)), both K-major,
// N >> 3 at [17,23), M >> 4 at [24,29), dense, no saturation.
__host__ __device__ constexpr uint32_t oz_idesc(int n) {
    return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(OZ_BM >> 4) << 24);
}

// Digits of four consecutive elements of a row in integer arithmetic: F = rint(a 2^(6 - e) 128^(S-1)) (|F| <= 2^(7S-1): one
// exact scaling and one rounding, the same residual |rho| <= 128^-(S-1) / 2 as S successive roundings), then the balanced
// base-128 digits of F read as bit fields of G = F + sum_j 64 128^j:  F = sum_j d_j 128^j, d_j = ((G >> 7j) & 127) - 64 in
// [-64, 63], the leading one (unmasked) in [-64, 64]; digit plane s holds q_s = d_(S-1-s).  (Successive rint / subtract /
// scale steps in FP64 cost ~150 instructions per element and made the pass issue-bound.)
struct OzDigitizer {
    int S, sh;
    double m1, m2;     // 2^sh = m1 m2, both always representable (|sh| <= 1130); x m1 m2 is exact wherever x 2^sh >= 1/2
    long long bias;
    int sq[OZ_MAX_S];  // sums of squared digits of the planes the diagonal correction needs (2 s >= S)
    __device__ __forceinline__ OzDigitizer(int S_, int e) : S(S_), sh(6 - e + 7 * (S_ - 1)) {
        m1 = ldexp(1.0, sh / 2);
        m2 = ldexp(1.0, sh - sh / 2);
        bias = 0;
        for (int jd = 0; jd < S; ++jd) bias += 64ll << (7 * jd);
#pragma unroll
        for (int s = 0; s < OZ_MAX_S; ++s) sq[s] = 0;
    }
    // four 7-bit fields of x -> four bytes (everything from bit 21 up goes to byte 3: the leading digit has 8 bits), then
    // field g = d + 64 -> the int8 d = (g + 64) ^ 0x80 in every byte at once (g + 64 <= 192: no carry between bytes)
    static __device__ __forceinline__ uint32_t fields_to_int8x4(uint32_t x) {
        const uint32_t w = (x & 0x7Fu) | ((x & 0x3F80u) << 1) | ((x & 0x1FC000u) << 2) | ((x & 0xFFE00000u) << 3);
        return (w + 0x40404040u) ^ 0x80808080u;
    }
    __device__ __forceinline__ void emit(const double (&x)[4], int8_t* dst, long long plane) {
        long long G[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) G[u] = __double2ll_rn(x[u] * m1 * m2) + bias;
        if (S == 8) {
            // 32-bit path: the low and the high 28 bits of G hold four digits each; bytes of an element's word = its
            // digits, a 4 x 4 byte transpose (PRMT) turns the words of four elements into the words of four planes
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t W[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    W[u] = fields_to_int8x4(h == 0 ? (uint32_t)G[u] & 0x0FFFFFFFu : (uint32_t)((unsigned long long)G[u] >> 28));
                const uint32_t t0 = __byte_perm(W[0], W[1], 0x5140), t1 = __byte_perm(W[2], W[3], 0x5140);
                const uint32_t t2 = __byte_perm(W[0], W[1], 0x7362), t3 = __byte_perm(W[2], W[3], 0x7362);
                uint32_t P[4];  // P[j]: digit 4 h + j (0 = least significant) of the four elements = plane 7 - (4 h + j)
                P[0] = __byte_perm(t0, t1, 0x5410);
                P[1] = __byte_perm(t0, t1, 0x7632);
                P[2] = __byte_perm(t2, t3, 0x5410);
                P[3] = __byte_perm(t2, t3, 0x7632);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int sp = 7 - (4 * h + j);
                    *reinterpret_cast<uint32_t*>(dst + (long long)sp * plane) = P[j];
                    if (h == 0) sq[sp] = __dp4a((int)P[j], (int)P[j], sq[sp]);   // planes 4..7 (2 s >= S)
                }
            }
            return;
        }
#pragma unroll
        for (int s = 0; s < OZ_MAX_S; ++s) {
            if (s < S) {
                const int pos = 7 * (S - 1 - s);
                int q[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) q[u] = (s == 0) ? (int)(G[u] >> pos) - 64 : ((int)(G[u] >> pos) & 127) - 64;
                *reinterpret_cast<char4*>(dst + (long long)s * plane) = make_char4((signed char)q[0], (signed char)q[1], (signed char)q[2], (signed char)q[3]);
                if (2 * s >= S) sq[s] += q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3];  // (N <= 65535: at most 64 x 4 x 4096 per thread)
            }
        }
    }
    __device__ __forceinline__ double corr() const {
        double w = 0.0;
#pragma unroll
        for (int s = 0; s < OZ_MAX_S; ++s)
            if (s < S && 2 * s >= S) w += ldexp((double)sq[s], -14 * s);
        return w;
    }
};

// ---------------------------------------------------------------------------------------------------
// Slicing: one block per row.  digits[s][row][k] (int8, row pitch kpad, zero beyond N), scale[row] = 2^{e_row}.
// ---------------------------------------------------------------------------------------------------
// corr[row] = sum_k sum_{2s >= S} 2^{-14 s} q_s[row][k]^2: the coherent part of the digit products the GEMM drops, for the
// DIAGONAL of an exact square A A^T.  Off the diagonal, between different matrices, and between different digit levels of
// one element, the dropped products are incoherent sums of magnitude sqrt(K) 2^{-7S}; on the diagonal of a square the
// s = t terms are sums of squares, a bias of K 64^2/3 2^{-7S}
// that the squaring chain T_2 -> T_4 -> ... -> T_k amplifies by 4 per doubling (measured at N = 5000, k = 32: |dtr D| = 9.5e-8
// without this term).  The epilogue adds it back when both factors are the same digit set.
__global__ void __launch_bounds__(256) oz_split_kernel(const double* __restrict__ A, long long lda, int N, int S, int8_t* __restrict__ digits,
                                                       long long kpad, double* __restrict__ scale, double* __restrict__ corr) {
    // one block per row (a row is read twice -- maximum, then digits -- and with a warp per row the rows in flight
    // exceeded the L2: measured 390 MB of DRAM reads for a 200 MB matrix)
    __shared__ double s_red[8];
    __shared__ int s_e;
    const int r = blockIdx.x, lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const double* row = A + (long long)r * lda;
    // 16-byte loads need an even leading dimension and an aligned base (plan-owned matrices; a caller's odd N falls back)
    const bool vec = ((lda & 1) == 0) && ((reinterpret_cast<uintptr_t>(A) & 15) == 0);
    double m = 0.0;
    if (vec) {
        for (int k = 2 * threadIdx.x; k < N; k += 512) {
            const double2 v = *reinterpret_cast<const double2*>(row + k);
            m = fmax(m, fabs(v.x));
            if (k + 1 < N) m = fmax(m, fabs(v.y));
        }
    } else {
        for (int k = threadIdx.x; k < N; k += 256) m = fmax(m, fabs(row[k]));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0) s_red[wid] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) m = fmax(m, s_red[q]);
        int e = 0;
        if (m > 0.0 && isfinite(m)) (void)frexp(m, &e);   // m = f 2^e, f in [0.5, 1)  =>  |a| 2^-e < 1
        s_e = e;
        scale[r] = ldexp(1.0, e);
    }
    __syncthreads();
    const int e = s_e;
    const long long plane = (long long)N * kpad;
    OzDigitizer dg(S, e);
    // four consecutive elements per thread and pass: whole 32-byte sectors per digit plane (kpad is a multiple of 64)
    for (long long k0 = 4 * threadIdx.x; k0 < kpad; k0 += 1024) {
        double x[4] = {0.0, 0.0, 0.0, 0.0};
        if (vec && k0 + 3 < N) {
            const double2 v0 = *reinterpret_cast<const double2*>(row + k0), v1 = *reinterpret_cast<const double2*>(row + k0 + 2);
            x[0] = v0.x; x[1] = v0.y; x[2] = v1.x; x[3] = v1.y;
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (k0 + u < N) x[u] = row[k0 + u];
        }
        dg.emit(x, digits + (long long)r * kpad + k0, plane);
    }
    double w = dg.corr();
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
    __syncthreads();
    if (lane == 0) s_red[wid] = w;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) w += s_red[q];
        corr[r] = w;
    }
}

// The same with the row held in registers between the two phases (kpad <= 1024 PASSES): every load of the row is in flight
// at once (a row per block and two dependent passes left ~24 KB per SM in flight: 0.37 of the HBM peak at N = 5000, and
// 4.5 waves of latency-bound blocks at N = 2000) and the row is read once.
template <int PASSES>
__global__ void __launch_bounds__(256) oz_split_reg_kernel(const double* __restrict__ A, long long lda, int N, int S, int8_t* __restrict__ digits,
                                                           long long kpad, double* __restrict__ scale, double* __restrict__ corr) {
    __shared__ double s_red[8];
    __shared__ int s_e;
    const int r = blockIdx.x, lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const double* row = A + (long long)r * lda;
    const bool vec = ((lda & 1) == 0) && ((reinterpret_cast<uintptr_t>(A) & 15) == 0);
    double x[PASSES][4];
#pragma unroll
    for (int i = 0; i < PASSES; ++i) {
        const int k0 = 4 * threadIdx.x + 1024 * i;
        if (vec && k0 + 3 < N) {
            const double2 v0 = *reinterpret_cast<const double2*>(row + k0), v1 = *reinterpret_cast<const double2*>(row + k0 + 2);
            x[i][0] = v0.x; x[i][1] = v0.y; x[i][2] = v1.x; x[i][3] = v1.y;
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u) x[i][u] = (k0 + u < N) ? row[k0 + u] : 0.0;
        }
    }
    double m = 0.0;
#pragma unroll
    for (int i = 0; i < PASSES; ++i)
#pragma unroll
        for (int u = 0; u < 4; ++u) m = fmax(m, fabs(x[i][u]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0) s_red[wid] = m;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) m = fmax(m, s_red[q]);
        int e = 0;
        if (m > 0.0 && isfinite(m)) (void)frexp(m, &e);
        s_e = e;
        scale[r] = ldexp(1.0, e);
    }
    __syncthreads();
    OzDigitizer dg(S, s_e);
    const long long plane = (long long)N * kpad;
#pragma unroll
    for (int i = 0; i < PASSES; ++i) {
        const long long k0 = 4 * threadIdx.x + 1024 * i;
        if (k0 < kpad) dg.emit(x[i], digits + (long long)r * kpad + k0, plane);
    }
    double w = dg.corr();
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) w += __shfl_xor_sync(0xffffffffu, w, o);
    __syncthreads();
    if (lane == 0) s_red[wid] = w;
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int q = 1; q < 8; ++q) w += s_red[q];
        corr[r] = w;
    }
}

struct OzArgs {
    int N, S;
    int kblocks;                 // kpad / OZ_BK
    int tiles_m, tiles_n;
    int sym;                     // 1: the product is symmetric (A and B commute): lower-triangle tiles only, mirrored on store
    int ntiles;                  // work items
    const short2* tile_list;     // [ntiles] (tm, tn) in raster order: column bands of OZ_BAND tiles, row-major inside a band, so
                                 // that the CTAs of a wave share few A and B digit strips (L2 reuse)
    const double* scaleA;        // [N] 2^{e_i}
    const double* scaleB;        // [N] 2^{f_j}
    const double* corr;          // nullable: [N] dropped-product sums of the diagonal (both factors are the same digit set)
    double alpha, beta;
    const double* C;             // nullable, leading dimension ldc
    long long ldc;
    const double* G;             // nullable: added with weight 1 (pre-formed low-order sum of Eq. 21), leading dimension ldg
    long long ldg;
    double diag;                 // added on the diagonal (- T_0 = - I of Eq. 22)
    double* Out;
    long long ldo;
};

template <int S>
__global__ void __launch_bounds__(OZ_THREADS, 1) oz_gemm_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                                                                const OzArgs args) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = smem_raw + ((1024u - (smem_u32(smem_raw) & 1023u)) & 1023u);
    const uint32_t ring_bytes = OZ_STAGES * OZ_MAX_S * (OZ_A_TILE + OZ_B_TILE);
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + ring_bytes);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + ring_bytes + 64);
    const uint32_t smem_base = smem_u32(smem);
    const uint32_t bar_base = smem_u32(bars);
    // (Releasing and refilling a stage in S sub-slots -- the A tile of digit s with the B tile of digit S-1-s, both dead
    // after the MMAs of digit s -- was measured 2.5 % SLOWER than whole-stage barriers: the kernel runs at the board's
    // power limit, SM clock ~1.78 GHz under ncu, not at a pipeline bubble.)
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (OZ_STAGES + s); };
    const uint32_t tfull_bar = bar_base + 8u * (2 * OZ_STAGES);
    const uint32_t tempty_bar = tfull_bar + 8u;
    const uint32_t stage_bytes = (uint32_t)S * (OZ_A_TILE + OZ_B_TILE);
    auto a_tile = [&](int stage, int s) { return smem_base + (uint32_t)stage * (OZ_MAX_S * (OZ_A_TILE + OZ_B_TILE)) + (uint32_t)s * OZ_A_TILE; };
    auto b_tile = [&](int stage, int t) { return smem_base + (uint32_t)stage * (OZ_MAX_S * (OZ_A_TILE + OZ_B_TILE)) + OZ_MAX_S * OZ_A_TILE + (uint32_t)t * OZ_B_TILE; };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int s = 0; s < OZ_STAGES; ++s) {
            mbar_init(full_bar(s), 1);
            mbar_init(empty_bar(s), 1);
        }
        mbar_init(tfull_bar, 1);
        mbar_init(tempty_bar, 8);   // the eight epilogue warps
        fence_mbar_init();
    }
    if (warp == 2) tc_alloc512(smem_u32(tmem_slot));
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int ntiles = args.ntiles;
    const int kblocks = args.kblocks;

    if (warp == 0) {
        // =================================== TMA producer ===================================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
                int tm, tn;
                tm = args.tile_list[t].x;
                tn = args.tile_list[t].y;
                for (int kb = 0; kb < kblocks; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1);
                    mbar_arrive_expect_tx(full_bar(stage), stage_bytes);
                    for (int s = 0; s < S; ++s) {
                        tma_load_3d(a_tile(stage, s), &mapA, full_bar(stage), kb * OZ_BK, tm * OZ_BM, s);
                        tma_load_3d(b_tile(stage, s), &mapB, full_bar(stage), kb * OZ_BK, tn * OZ_BN, s);
                    }
                    if (++stage == OZ_STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // =================================== MMA issuer ===================================
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0, tphase = 0;
            for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
                mbar_wait(tempty_bar, tphase ^ 1);   // the epilogue has drained the accumulators of the previous tile
                tc_fence_after();
                for (int kb = 0; kb < kblocks; ++kb) {
                    mbar_wait(full_bar(stage), phase);
                    tc_fence_after();
                    // Digit s of A meets the digits q = 0 .. S-1-s of B, whose tiles are consecutive in shared memory (64 rows
                    // each) and whose accumulators d = s + q are consecutive in tensor memory (64 columns each): one MMA of
                    // N = 64 (S - s) columns (two when that exceeds 256) instead of S - s MMAs of N = 64 -- the single issuing
                    // thread cannot feed 32-cycle MMAs fast enough (measured: 1.6 POPS with N = 64, see profiles/).
#pragma unroll
                    for (int s = 0; s < S; ++s) {
                        const uint64_t ad = oz_smem_desc(a_tile(stage, s));
                        const int nq = S - s;                          // digits of B
                        const int n0 = (nq > 4) ? 4 : nq;              // first MMA: up to 4 digits (N <= 256)
#pragma unroll
                        for (int kk = 0; kk < OZ_BK / 32; ++kk) {
                            // first touch of every accumulator of a tile: k-block 0, s = 0, first K = 32 step
                            const uint32_t acc = (kb > 0 || s > 0 || kk > 0) ? 1u : 0u;
                            const uint64_t koff = (uint64_t)(kk * 32 >> 4);
                            tc_mma_i8(tmem_base + (uint32_t)s * OZ_BN, ad + koff, oz_smem_desc(b_tile(stage, 0)) + koff, oz_idesc(64 * n0), acc);
                            if (nq > 4)
                                tc_mma_i8(tmem_base + (uint32_t)(s + 4) * OZ_BN, ad + koff, oz_smem_desc(b_tile(stage, 4)) + koff,
                                          oz_idesc(64 * (nq - 4)), acc);
                        }
                    }
                    tc_commit(empty_bar(stage));                   // stage back to the producer when these MMAs are done
                    if (++stage == OZ_STAGES) { stage = 0; phase ^= 1; }
                }
                tc_commit(tfull_bar);                              // accumulators complete
                tphase ^= 1;
            }
        }
    } else if (warp >= 4) {
        // =================================== epilogue warps ===================================
        // eight epilogue warps: two per TMEM lane quarter (a warp may only access the quarter warp % 4), each taking half of
        // the 64 columns -- the epilogue is a chain of latencies (tcgen05.ld, the C / G tiles from L2, stores) that holds the
        // tensor pipe up (all 512 TMEM columns are in use: no second accumulator set to overlap with); measured with four warps:
        // ~17 us of a 77 us tile at N = 2000
        const int q4 = warp & 3;                                   // TMEM lane quarter this warp may access
        const int chalf = (warp - 4) >> 2;                         // column half
        const uint32_t lane_base = tmem_base + ((uint32_t)(q4 * 32) << 16);
        uint32_t tphase = 0;
        const int N = args.N;
        for (int t = blockIdx.x; t < ntiles; t += gridDim.x) {
            int tm, tn;
            tm = args.tile_list[t].x;
            tn = args.tile_list[t].y;
            mbar_wait(tfull_bar, tphase);
            tphase ^= 1;
            tc_fence_after();
            const int row = tm * OZ_BM + q4 * 32 + lane;
            const bool vecC = (args.C == nullptr) || (((args.ldc & 1) == 0) && ((reinterpret_cast<uintptr_t>(args.C) & 15) == 0));
            const bool vecG = (args.G == nullptr) || (((args.ldg & 1) == 0) && ((reinterpret_cast<uintptr_t>(args.G) & 15) == 0));
            const bool vecS = (reinterpret_cast<uintptr_t>(args.scaleB) & 15) == 0;
            const bool vecO = ((args.ldo & 1) == 0) && ((reinterpret_cast<uintptr_t>(args.Out) & 15) == 0);
            const double rs = (row < N) ? args.scaleA[row] * args.alpha * (1.0 / 4096.0) : 0.0;   // alpha 2^{e_i - 12}
            for (int c8 = chalf * (OZ_BN / 16); c8 < (chalf + 1) * (OZ_BN / 16); ++c8) {
                const int col0 = tn * OZ_BN + c8 * 8;
                // the C / G / scale operands of the chunk are requested before the accumulators are read from tensor memory
                double cv[8], gv[8], sb[8];
                if (row < N && col0 + 7 < N && vecC && vecG && vecS) {   // whole chunk inside, 16-byte aligned rows: 128-bit loads
#pragma unroll
                    for (int j = 0; j < 8; j += 2) {
                        const double2 s2 = *reinterpret_cast<const double2*>(args.scaleB + col0 + j);
                        sb[j] = s2.x; sb[j + 1] = s2.y;
                        double2 c2 = make_double2(0.0, 0.0), g2 = make_double2(0.0, 0.0);
                        if (args.C != nullptr) c2 = *reinterpret_cast<const double2*>(args.C + (long long)row * args.ldc + col0 + j);
                        if (args.G != nullptr) g2 = *reinterpret_cast<const double2*>(args.G + (long long)row * args.ldg + col0 + j);
                        cv[j] = c2.x; cv[j + 1] = c2.y;
                        gv[j] = g2.x; gv[j + 1] = g2.y;
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < 8; ++j) {
                        const int col = col0 + j;
                        const bool in = (row < N && col < N);
                        sb[j] = in ? args.scaleB[col] : 0.0;
                        cv[j] = (in && args.C != nullptr) ? args.C[(long long)row * args.ldc + col] : 0.0;
                        gv[j] = (in && args.G != nullptr) ? args.G[(long long)row * args.ldg + col] : 0.0;
                    }
                }
                int v[S][8];
#pragma unroll
                for (int d = 0; d < S; ++d) tc_ld8(lane_base + (uint32_t)(d * OZ_BN + c8 * 8), v[d]);
                tc_wait_ld();
                double r[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) r[j] = 0.0;
#pragma unroll
                for (int d = S - 1; d >= 0; --d)                   // Horner from the least significant digit sum
#pragma unroll
                    for (int j = 0; j < 8; ++j) r[j] = fma(r[j], 1.0 / 128.0, (double)v[d][j]);
                double ov[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int col = col0 + j;
                    if (args.corr != nullptr && row == col && row < N) r[j] += args.corr[row];
                    double o = rs * sb[j] * r[j];
                    o = fma(args.beta, cv[j], o);
                    o += gv[j];
                    if (row == col) o += args.diag;
                    ov[j] = o;
                }
                const bool whole = vecO && row < N && col0 + 7 < N;
                if (whole) {
#pragma unroll
                    for (int j = 0; j < 8; j += 2)
                        *reinterpret_cast<double2*>(args.Out + (long long)row * args.ldo + col0 + j) = make_double2(ov[j], ov[j + 1]);
                }
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                    const int col = col0 + j;
                    if (row < N && col < N) {
                        const double o = ov[j];
                        if (!whole) args.Out[(long long)row * args.ldo + col] = o;
                        // mirror: the transposed element lies in a tile that is not a work item; the lanes of a warp hold 32
                        // consecutive rows, i.e. 32 consecutive elements of the destination row: coalesced
                        if (args.sym && (col / OZ_BM) * OZ_BM + OZ_BM - 1 < (row / OZ_BN) * OZ_BN) args.Out[(long long)col * args.ldo + row] = o;
                    }
                }
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive(tempty_bar);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 2) {
        tc_fence_after();
        tc_dealloc512(tmem_base);
    }
}

inline int oz_smem_bytes() { return OZ_STAGES * OZ_MAX_S * (OZ_A_TILE + OZ_B_TILE) + 128 + 1024; }

}  // namespace chebdm
