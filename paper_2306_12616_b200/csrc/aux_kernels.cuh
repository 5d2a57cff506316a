// aux_kernels.cuh -- the non-GEMM kernels of the hot path (sm_100a): Gershgorin bounds fused with the
// affine rescale (north_star item 1), the device-side coefficient pipeline (c_n by DCT, then the g/d
// tables of Eq. 16-20), trace / mu search (north_star item 4).  Product code; shares nothing with oracle/.
#pragma once
#include <cooperative_groups.h>
#include "common.cuh"

namespace chebdm {
namespace cg = cooperative_groups;

// ---------------------------------------------------------------------------------------------------
// Device-resident scalar state of one matrix ("slot") of a plan.
// ---------------------------------------------------------------------------------------------------
struct DevScalars {
    double a, b;                      // bounds in use (eps_a, eps_b)
    int bad_bounds;                   // sticky: set when the bounds are non-finite; cleared by cheb_dm_check
    int noconv;                       // sticky: the power-basis table d of Eq. (4) exceeded the stability guard
    double mu;                        // chemical potential in use (given, or the result of the device-side bisection)
    double ne;                        // N_e at that mu (bisection only)
};

// Copy a user matrix (ld N) into a padded workspace matrix (ld ldx).
__global__ void pad_copy_kernel(const double* __restrict__ src, long long lds, int N, double* __restrict__ dst, long long ldx) {
    const long long total = (long long)N * N;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(e / N), j = (int)(e - (long long)i * N);
        dst[(long long)i * ldx + j] = src[(long long)i * lds + j];
    }
}
__global__ void unpad_copy_kernel(const double* __restrict__ src, long long ldx, int N, double* __restrict__ dst, long long ldd) {
    const long long total = (long long)N * N;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(e / N), j = (int)(e - (long long)i * N);
        dst[(long long)i * ldd + j] = src[(long long)i * ldx + j];
    }
}

// The same for a symmetric source of which only the symBM x symBN tiles that touch the lower triangle were formed
// (form_sums with symmetric-tile skipping): an element of a skipped tile is read from its mirror image, which lies
// strictly below the diagonal and therefore in a formed tile.
__global__ void unpad_copy_sym_kernel(const double* __restrict__ src, long long ldx, int N, double* __restrict__ dst, long long ldd,
                                      int symBM, int symBN) {
    const long long total = (long long)N * N;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < total; e += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(e / N), j = (int)(e - (long long)i * N);
        const bool skipped = (i / symBM) * symBM + symBM - 1 < (j / symBN) * symBN;
        dst[(long long)i * ldd + j] = skipped ? src[(long long)j * ldx + i] : src[(long long)i * ldx + j];
    }
}

// ---------------------------------------------------------------------------------------------------
// Double-double helpers (error-free transformations) for the scalar reductions: the parity gate on D
// needs sum_n |delta c_n| << 1e-10 with N_q up to 8192 quadrature terms per coefficient.
// ---------------------------------------------------------------------------------------------------
struct dd { double hi, lo; };
__device__ __forceinline__ dd dd_add_prod(dd s, double x, double y) {  // s + x*y
    const double p = x * y;
    const double e = fma(x, y, -p);
    const double t = s.hi + p;
    const double bb = t - s.hi;
    const double err = (s.hi - (t - bb)) + (p - bb);
    dd r;
    r.hi = t;
    r.lo = s.lo + err + e;
    return r;
}
__device__ __forceinline__ dd dd_add(dd x, dd y) {
    const double t = x.hi + y.hi;
    const double bb = t - x.hi;
    const double err = (x.hi - (t - bb)) + (y.hi - bb);
    dd r;
    r.hi = t;
    r.lo = x.lo + y.lo + err;
    return r;
}
// Fixed-order block reduction of a dd (blockDim.x <= 1024, multiple of 32). Result valid in thread 0.
__device__ __forceinline__ dd dd_block_reduce(dd v, dd* s_buf) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dd other;
        other.hi = __shfl_down_sync(0xffffffffu, v.hi, o);
        other.lo = __shfl_down_sync(0xffffffffu, v.lo, o);
        v = dd_add(v, other);
    }
    if (lane == 0) s_buf[warp] = v;
    __syncthreads();
    if (warp == 0) {
        const int nw = blockDim.x >> 5;
        v.hi = lane < nw ? s_buf[lane].hi : 0.0;
        v.lo = lane < nw ? s_buf[lane].lo : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            dd other;
            other.hi = __shfl_down_sync(0xffffffffu, v.hi, o);
            other.lo = __shfl_down_sync(0xffffffffu, v.lo, o);
            v = dd_add(v, other);
        }
    }
    __syncthreads();
    return v;
}

// Fermi function of the scaled variable, overflow-safe (Eq. 2).
__device__ __forceinline__ double fermi_scaled(double beta_t, double mu_t, double x) {
    const double y = beta_t * (x - mu_t);
    if (y > 0.0) {
        const double e = exp(-y);
        return e / (1.0 + e);
    }
    return 1.0 / (1.0 + exp(y));
}

// ---------------------------------------------------------------------------------------------------
// a-1 .. a-3 fused: ONE cooperative launch does everything that precedes the products, for every matrix of the batch.
// Block b serves matrix (slot) b % nb; the blocks of a slot split its rows / nodes / coefficients among themselves.
//   phase 0  zero the scheduler counters (replaces a memset node); the sticky error flag lies outside that range
//   phase 1  (do_bounds) Gershgorin: one warp per row, per-block (min, max) partials -- no atomics, so no
//            initialisation pass and a result that does not depend on the order of arrival
//   -- grid sync --
//   phase 2  every block reduces its slot's partials to (a, b) itself; rescale H -> X = T_1 (pad columns stay zero);
//            (do_coeffs) fn[j] = f~(x_j) at the N_q Chebyshev nodes, mu given per slot or read from the slot's
//            DevScalars (mu_from_device: the result of the device-side bisection, cheb_dm_solve)
//   -- grid sync --
//   phase 3  c_n, n < k p: one warp per coefficient, double-double accumulation in a fixed order
//   -- grid sync --
//   phase 4  (first block of the slot) tables g (and d) of Eq. (16)-(20).  Thread i owns the coupled chains i and
//            k-i of g_{i,l} = 2 c_{lk+i} - g_{k-i,l+1}, so the recurrence needs no block barrier.  With the power-basis
//            outer recursion (want_d) the guard of reading A6 is evaluated: max|d| 2^-52 p > 1e-12 sets `noconv`
//            (d_{i,p-1} = 2^p c by Eq. 12's a_{j,j} = 2^{1-j}).
// do_bounds = 0, do_coeffs = 1 recomputes the tables only (new mu on the same X: cheb_dm_solve, cheb_dm_remu).
// For small N the launch gaps of five separate kernels were ~10 % of a whole solve (cfg1: 39 us of 400 us).
// HBM bytes: 8N^2 read (+ 8N^2 re-read, L2 for small N) + 8N^2 written per matrix.
// ---------------------------------------------------------------------------------------------------
constexpr int FRONT_SMEM_COEFS = 4608;  // 36 KB: covers k p up to 4608 (all configs; larger plans read c from L2)
struct FrontArgs {
    int nb;                          // matrices of this call (gridDim.x >= nb)
    int N;
    const double* H[MAX_BATCH];      // per slot, leading dimension ldh
    double mu[MAX_BATCH];            // per slot (ignored when mu_from_device)
    long long ldh;
    double* X;                       // T_1 of slot 0; slot s at X + s * slot_stride
    long long slot_stride, ldx;
    DevScalars* sc;                  // [nb]
    int explicit_bounds;
    double a, b;                     // explicit bounds
    double* part;                    // [2 * gridDim.x] per-block (lo, hi)
    int* counters;                   // range to zero
    int ncounters;
    int do_bounds, do_coeffs, mu_from_device;
    int segs;                        // warps of a block that share a row in the bounds / rescale passes (1, 2, 4, 8 or 16)
    double beta;
    const double* costab;
    int Nq, M;
    double* fn;                      // [slot][Nq]
    double* c;                       // [slot][k p]
    int k, p;
    const double* Amat;
    int want_d;
    double* gT;                      // [slot][p][k]
    double* dT;
};

__global__ void __launch_bounds__(512) front_end_kernel(const FrontArgs A) {
    cg::grid_group grid = cg::this_grid();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int warps_per_block = blockDim.x >> 5;
    const int nb = A.nb;
    const int slot = blockIdx.x % nb, sblock = blockIdx.x / nb;
    const int sblocks = ((int)gridDim.x - slot + nb - 1) / nb;          // blocks that serve this slot
    const int gwarp = sblock * warps_per_block + warp, nwarps = sblocks * warps_per_block;
    const int N = A.N;
    const int kp = A.k * A.p;
    const double* __restrict__ H = A.H[slot];
    const long long ldh = A.ldh;
    DevScalars* sc = A.sc + slot;
    __shared__ double s_lo[32], s_hi[32];
    __shared__ double s_ab[2];
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < A.ncounters; e += gridDim.x * blockDim.x) A.counters[e] = 0;
    double a, b;
    if (A.do_bounds) {
        const bool vec = ((ldh & 1) == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
        if (!A.explicit_bounds) {
            double lo = INFINITY, hi = -INFINITY;
            // `segs` consecutive warps of a block share a row (segment seg = columns [seg seglen, (seg+1) seglen)); their
            // partial sums are combined in a fixed order through shared memory.  segs = 1 for small N (a warp per row);
            // for N = 5000 a warp per row left 264 rows for a second round (2 x 79 serial iterations per warp).
            const int segs = A.segs, rpb = warps_per_block / segs;          // rows per block and round
            const int seg = warp % segs, rloc = warp / segs;
            const int seglen = (((N + segs - 1) / segs) + 1) & ~1;           // even: 16-byte loads stay aligned
            const int j0 = seg * seglen, j1 = min(N, j0 + seglen);
            for (int rbase = sblock * rpb; rbase < N; rbase += sblocks * rpb) {
                const int row = rbase + rloc;
                double r = 0.0, hii = 0.0;
                if (row < N) {
                    const double* hr = H + (long long)row * ldh;
                    if (vec) {
                        // pairs [j, j+1] below jend, four 16-byte loads in flight per lane; an odd last column apart
                        const int jend = j1 & ~1;
                        int j = j0 + 2 * lane;
                        for (; j + 192 < jend; j += 256) {
                            double2 v[4];
#pragma unroll
                            for (int u = 0; u < 4; ++u) v[u] = __ldg(reinterpret_cast<const double2*>(hr + j + 64 * u));
#pragma unroll
                            for (int u = 0; u < 4; ++u) {
                                if (j + 64 * u == row) hii = v[u].x; else r += fabs(v[u].x);
                                if (j + 64 * u + 1 == row) hii = v[u].y; else r += fabs(v[u].y);
                            }
                        }
                        for (; j < jend; j += 64) {
                            const double2 v = __ldg(reinterpret_cast<const double2*>(hr + j));
                            if (j == row) hii = v.x; else r += fabs(v.x);
                            if (j + 1 == row) hii = v.y; else r += fabs(v.y);
                        }
                        if ((j1 & 1) && j0 < j1 && lane == 0) {
                            const double v = hr[j1 - 1];
                            if (j1 - 1 == row) hii = v; else r += fabs(v);
                        }
                    } else {
                        for (int j = j0 + lane; j < j1; j += 32) {
                            const double v = hr[j];
                            if (j == row) hii = v; else r += fabs(v);
                        }
                    }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    r += __shfl_xor_sync(0xffffffffu, r, o);
                    hii += __shfl_xor_sync(0xffffffffu, hii, o);  // exactly one lane of one segment holds h_ii, the rest 0
                }
                if (segs > 1) {
                    if (lane == 0) { s_lo[warp] = r; s_hi[warp] = hii; }   // (s_lo / s_hi double as the segment scratch here)
                    __syncthreads();
                    if (seg == 0) {
                        r = 0.0;
                        hii = 0.0;
                        for (int q = 0; q < segs; ++q) { r += s_lo[warp + q]; hii += s_hi[warp + q]; }
                    }
                    __syncthreads();
                }
                if (seg == 0 && row < N) {
                    lo = fmin(lo, hii - r);
                    hi = fmax(hi, hii + r);
                    if (!(isfinite(r) && isfinite(hii))) { lo = -INFINITY; hi = INFINITY; }
                }
            }
            if (lane == 0) { s_lo[warp] = lo; s_hi[warp] = hi; }
            __syncthreads();
            if (warp == 0) {
                lo = lane < warps_per_block ? s_lo[lane] : INFINITY;
                hi = lane < warps_per_block ? s_hi[lane] : -INFINITY;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
                    hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
                }
                if (lane == 0) {
                    A.part[2 * blockIdx.x] = lo;
                    A.part[2 * blockIdx.x + 1] = hi;
                }
            }
            grid.sync();
            if (warp == 0) {
                lo = INFINITY;
                hi = -INFINITY;
                for (int bIdx = slot + nb * lane; bIdx < (int)gridDim.x; bIdx += 32 * nb) {  // the blocks of this slot
                    lo = fmin(lo, __ldcg(A.part + 2 * bIdx));
                    hi = fmax(hi, __ldcg(A.part + 2 * bIdx + 1));
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
                    hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
                }
                if (lane == 0) {
                    s_ab[0] = lo;
                    s_ab[1] = hi;
                }
            }
            __syncthreads();
        } else if (threadIdx.x == 0) {
            s_ab[0] = A.a;
            s_ab[1] = A.b;
        }
        __syncthreads();
        a = s_ab[0];
        b = s_ab[1];
        const bool bad = !(isfinite(a) && isfinite(b));
        if (a == b) { a -= 1.0; b += 1.0; }  // degenerate H = cI (reading A2-iv)
        if (sblock == 0 && threadIdx.x == 0) {
            sc->a = a;
            sc->b = b;
            if (bad) sc->bad_bounds = 1;  // sticky
        }
        // ---- phase 2: rescale ----
        const double inv = 1.0 / (b - a), shift = a + b;
        double* X = A.X + (long long)slot * A.slot_stride;
        {
            const int segs = A.segs, rpb = warps_per_block / segs;
            const int seg = warp % segs, rloc = warp / segs;
            const int seglen = (((N + segs - 1) / segs) + 1) & ~1;
            const int j0 = seg * seglen, j1 = min(N, j0 + seglen);
            for (int rbase = sblock * rpb; rbase < N; rbase += sblocks * rpb) {
                const int row = rbase + rloc;
                if (row >= N) continue;
                const double* hr = H + (long long)row * ldh;
                double* xr = X + (long long)row * A.ldx;
                if (vec) {
                    const int jend = j1 & ~1;
                    int j = j0 + 2 * lane;
                    for (; j + 192 < jend; j += 256) {
                        double2 v[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) v[u] = __ldg(reinterpret_cast<const double2*>(hr + j + 64 * u));
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            double h0 = 2.0 * v[u].x, h1 = 2.0 * v[u].y;
                            if (j + 64 * u == row) h0 -= shift;
                            if (j + 64 * u + 1 == row) h1 -= shift;
                            *reinterpret_cast<double2*>(xr + j + 64 * u) = make_double2(h0 * inv, h1 * inv);
                        }
                    }
                    for (; j < jend; j += 64) {
                        const double2 v = __ldg(reinterpret_cast<const double2*>(hr + j));
                        double h0 = 2.0 * v.x, h1 = 2.0 * v.y;
                        if (j == row) h0 -= shift;
                        if (j + 1 == row) h1 -= shift;
                        *reinterpret_cast<double2*>(xr + j) = make_double2(h0 * inv, h1 * inv);
                    }
                    if ((j1 & 1) && j0 < j1 && lane == 0) {
                        double h = 2.0 * hr[j1 - 1];
                        if (j1 - 1 == row) h -= shift;
                        xr[j1 - 1] = h * inv;
                    }
                } else {
                    for (int j = j0 + lane; j < j1; j += 32) {
                        double h = 2.0 * hr[j];
                        if (j == row) h -= shift;
                        xr[j] = h * inv;
                    }
                }
            }
        }
    } else {
        a = __ldcg(&sc->a);
        b = __ldcg(&sc->b);
    }
    if (!A.do_coeffs) return;
    double* fn = A.fn + (size_t)slot * A.Nq;
    double* c = A.c + (size_t)slot * kp;
    {
        const double mu = A.mu_from_device ? __ldcg(&sc->mu) : A.mu[slot];
        if (!A.mu_from_device && sblock == 0 && threadIdx.x == 0) sc->mu = mu;
        const double beta_t = A.beta * (b - a) * 0.5;
        const double mu_t = (2.0 * mu - (a + b)) / (b - a);
        for (int j = sblock * blockDim.x + threadIdx.x; j < A.Nq; j += sblocks * blockDim.x)
            fn[j] = fermi_scaled(beta_t, mu_t, A.costab[2 * j + 1]);
    }
    grid.sync();
    // ---- phase 3: c_n (one warp per coefficient) ----
    {
        const unsigned mask = 4u * (unsigned)A.Nq - 1u;
        for (int n = gwarp; n < kp; n += nwarps) {
            double cn = 0.0;
            if (n < A.M) {
                dd s;
                s.hi = 0.0;
                s.lo = 0.0;
                for (int j = lane; j < A.Nq; j += 32) {
                    const unsigned r = ((unsigned)n * (2u * (unsigned)j + 1u)) & mask;
                    s = dd_add_prod(s, __ldcg(fn + j), A.costab[r]);
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    dd other;
                    other.hi = __shfl_down_sync(0xffffffffu, s.hi, o);
                    other.lo = __shfl_down_sync(0xffffffffu, s.lo, o);
                    s = dd_add(s, other);
                }
                cn = ((n == 0) ? 1.0 : 2.0) * (s.hi + s.lo) / (double)A.Nq;
            }
            if (lane == 0) c[n] = cn;
        }
    }
    grid.sync();
    // ---- phase 4: tables (first block of the slot).  Layout gT[l*k + i], dT likewise ----
    if (sblock != 0) return;
    {
        const int k = A.k, p = A.p;
        double* gT = A.gT + (size_t)slot * kp;
        double* dT = A.dT + (size_t)slot * kp;
        // stage c in shared memory when it fits (one coalesced pass instead of 2p dependent L2 round trips per thread)
        __shared__ double s_c[FRONT_SMEM_COEFS];
        __shared__ unsigned long long s_dmax;
        const bool staged = (kp <= FRONT_SMEM_COEFS);
        if (threadIdx.x == 0) s_dmax = 0ull;
        if (staged) {
            for (int e = threadIdx.x; e < kp; e += blockDim.x) s_c[e] = __ldcg(c + e);
        }
        __syncthreads();
        const double* cc = staged ? s_c : c;
        for (int l = threadIdx.x; l < p; l += blockDim.x) gT[(size_t)l * k] = cc[(size_t)l * k];
        // pairs (i, k-i), 1 <= i <= k/2 (i == k-i when k is even and i = k/2)
        for (int i = 1 + threadIdx.x; 2 * i <= k; i += blockDim.x) {
            const int i2 = k - i;
            double g1 = 0.0, g2 = 0.0;  // g_{i,l+1}, g_{k-i,l+1}
            for (int l = p - 1; l >= 0; --l) {
                const double c1 = cc[(size_t)l * k + i], c2 = cc[(size_t)l * k + i2];
                double n1, n2;
                if (p == 1) { n1 = c1; n2 = c2; }
                else if (l == p - 1) { n1 = 2.0 * c1; n2 = 2.0 * c2; }
                else if (l >= 1) { n1 = 2.0 * c1 - g2; n2 = 2.0 * c2 - g1; }
                else { n1 = c1 - 0.5 * g2; n2 = c2 - 0.5 * g1; }
                gT[(size_t)l * k + i] = n1;
                gT[(size_t)l * k + i2] = n2;
                g1 = n1;
                g2 = n2;
            }
        }
        if (A.want_d) {
            __syncthreads();
            double dmax = 0.0;
            for (int i = threadIdx.x; i < k; i += blockDim.x) {
                for (int l = p - 1; l >= 0; --l) {
                    double s = gT[(size_t)l * k + i];
                    for (int j = l + 1; j < p; ++j) s -= A.Amat[(size_t)j * p + l] * dT[(size_t)j * k + i];
                    const double d = s / A.Amat[(size_t)l * p + l];
                    dT[(size_t)l * k + i] = d;
                    dmax = fmax(dmax, fabs(d));
                }
            }
            if (!(dmax <= 1.7e308)) dmax = 1.7e308;  // NaN / inf trip the guard too
            atomicMax(&s_dmax, (unsigned long long)__double_as_longlong(dmax));  // non-negative doubles order like integers
            __syncthreads();
            if (threadIdx.x == 0) {
                const double m = __longlong_as_double((long long)s_dmax);
                if (m * 2.220446049250313e-16 * (double)p > 1e-12) sc->noconv = 1;  // sticky (reading A6)
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// a-7: trace.  One block per matrix, fixed summation order (bitwise reproducible).  8N useful bytes each.
// ---------------------------------------------------------------------------------------------------
struct TraceArgs {
    const double* D[MAX_BATCH];
};
__global__ void __launch_bounds__(1024) trace_kernel(const TraceArgs A, int N, long long ld, double* __restrict__ out) {
    __shared__ dd s_buf[32];
    const double* __restrict__ D = A.D[blockIdx.x];
    dd s;
    s.hi = 0.0;
    s.lo = 0.0;
    for (int i = threadIdx.x; i < N; i += blockDim.x) s = dd_add_prod(s, D[(long long)i * ld + i], 1.0);
    s = dd_block_reduce(s, s_buf);
    if (threadIdx.x == 0) out[blockIdx.x] = s.hi + s.lo;
}

// ---------------------------------------------------------------------------------------------------
// a-7: moments tau_n = tr T_n(X), n < k p (reading A10).  With U_j = T_j(T_k) = T_{jk}(X):
//     tau_i = tr T_i (i <= k),  tau_{jk} = tr U_j,  tau_{jk+i} = 2 <U_j, T_i>_F - tau_{jk-i}   (Eq. 7 + symmetry).
// The baby block T_1..T_k and the giant block U_2..U_{p-1} are resident in the workspace (U_1 = T_k), so all inner
// products are ONE skinny GEMM over the matrix elements,  Gram[j][i] = sum_e U_j[e] T_i[e]  (K = N ld elements),
// which reads every matrix once per 32 x 32 block of the Gram matrix instead of k-1 matrices per product epilogue.
//   diag_traces_kernel: block (m, slot): trace of the m-th workspace matrix (T_1..T_k, then U_2..U_{p-1})
//   gram_kernel       : grid (CTAs, passes, slots); a pass is one 32 x 32 block (rb, cb) of the Gram matrix; every warp
//                       owns a contiguous range of 8-element chunks and accumulates its 32 x 32 partial on the tensor
//                       cores (DMMA.8x8x4: lane (g, t) feeds element pair 2t, 2t+1 of row-matrix g and column-matrix g);
//                       the 8 warps are added in a fixed order, one partial per CTA
//   moments_kernel    : one block per slot: sums the CTA partials in a fixed order, then the tau recurrence
// Pad columns of every workspace matrix are zero, so the padded elements contribute nothing.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) diag_traces_kernel(const double* __restrict__ Tbase, const double* __restrict__ Ubase,
                                                          long long stride, long long slot_stride, long long ld, int N, int k,
                                                          double* __restrict__ traces, int nmat) {
    __shared__ dd s_buf[32];
    const int m = blockIdx.x, slot = blockIdx.y;
    const double* Mx = (m < k ? Tbase + (long long)m * stride : Ubase + (long long)(m - k) * stride) + (long long)slot * slot_stride;
    dd s;
    s.hi = 0.0;
    s.lo = 0.0;
    for (int r = threadIdx.x; r < N; r += blockDim.x) s = dd_add_prod(s, Mx[(long long)r * ld + r], 1.0);
    s = dd_block_reduce(s, s_buf);
    if (threadIdx.x == 0) traces[(size_t)slot * nmat + m] = s.hi + s.lo;
}

constexpr int GRAM_BLK = 32;
// NB = 8-row blocks per side actually formed (4: a full 32 x 32 block of the Gram matrix; 2 or 1 when p - 1 and k - 1 are at
// most 16 or 8: the padded blocks would cost as many DMMAs as the needed ones and make the pass tensor-bound)
template <int NB>
__global__ void __launch_bounds__(256) gram_kernel(const double* __restrict__ Tbase, const double* __restrict__ Ubase, long long stride,
                                                   long long slot_stride, long long nelem, int k, int p,
                                                   double* __restrict__ partial /* [slot][pass][cta][32*32] */) {
    __shared__ double s_acc[GRAM_BLK * GRAM_BLK];
    const int R = p - 1, Cn = k - 1;                       // Gram rows (U_1..U_{p-1}) and columns (T_1..T_{k-1})
    const int npc = (Cn + GRAM_BLK - 1) / GRAM_BLK;
    const int rb = blockIdx.y / npc, cb = blockIdx.y - rb * npc;
    const int slot = blockIdx.z;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const double* Ts = Tbase + (long long)slot * slot_stride;
    const double* Us = Ubase + (long long)slot * slot_stride;
    const double* rowp[NB];
    const double* colp[NB];
    bool rowv[NB], colv[NB];
#pragma unroll
    for (int mb = 0; mb < NB; ++mb) {
        const int r = rb * GRAM_BLK + mb * 8 + g;
        rowv[mb] = r < R;
        rowp[mb] = (r == 0 || !rowv[mb]) ? Ts + (long long)(k - 1) * stride : Us + (long long)(r - 1) * stride;  // U_1 = T_k
        const int q = cb * GRAM_BLK + mb * 8 + g;
        colv[mb] = q < Cn;
        colp[mb] = Ts + (long long)(colv[mb] ? q : 0) * stride;
    }
    double acc[NB][NB][2];
#pragma unroll
    for (int i = 0; i < NB; ++i)
#pragma unroll
        for (int j = 0; j < NB; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const long long nchunks = nelem / 8;                  // nelem = N ld, ld a multiple of 16
    const long long W = (long long)gridDim.x * 8, w = (long long)blockIdx.x * 8 + warp;
    const long long per = (nchunks + W - 1) / W;
    const long long c0 = w * per, c1 = (c0 + per < nchunks) ? c0 + per : nchunks;
#pragma unroll 2
    for (long long ch = c0; ch < c1; ++ch) {
        const long long e = ch * 8 + 2 * t;
        double2 a[NB], b[NB];
#pragma unroll
        for (int mb = 0; mb < NB; ++mb) {
            a[mb] = rowv[mb] ? __ldcs(reinterpret_cast<const double2*>(rowp[mb] + e)) : make_double2(0.0, 0.0);
            b[mb] = colv[mb] ? __ldcs(reinterpret_cast<const double2*>(colp[mb] + e)) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int i = 0; i < NB; ++i)
#pragma unroll
            for (int j = 0; j < NB; ++j) {
                dmma_884(acc[i][j][0], acc[i][j][1], a[i].x, b[j].x);
                dmma_884(acc[i][j][0], acc[i][j][1], a[i].y, b[j].y);
            }
    }
    // fixed-order sum of the 8 warps (each lane owns distinct entries), one partial per CTA
    for (int e = threadIdx.x; e < GRAM_BLK * GRAM_BLK; e += blockDim.x) s_acc[e] = 0.0;
    __syncthreads();
    for (int wv = 0; wv < 8; ++wv) {
        if (warp == wv) {
#pragma unroll
            for (int i = 0; i < NB; ++i)
#pragma unroll
                for (int j = 0; j < NB; ++j) {
                    s_acc[(i * 8 + g) * GRAM_BLK + j * 8 + 2 * t] += acc[i][j][0];
                    s_acc[(i * 8 + g) * GRAM_BLK + j * 8 + 2 * t + 1] += acc[i][j][1];
                }
        }
        __syncthreads();
    }
    double* dst = partial + (((size_t)slot * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * (GRAM_BLK * GRAM_BLK);
    for (int e = threadIdx.x; e < GRAM_BLK * GRAM_BLK; e += blockDim.x) dst[e] = s_acc[e];
}

// traces: [slot][nmat] (T_1..T_k, U_2..U_{p-1}); partial: gram_kernel's output; gram: scratch [slot][(p-1)(k-1)].
__global__ void __launch_bounds__(1024) moments_kernel(const double* __restrict__ traces, int nmat, const double* __restrict__ partial,
                                                      int nctas, int npasses, double* __restrict__ gram, int k, int p, int N,
                                                      double* __restrict__ tau_all) {
    const int slot = blockIdx.x;
    const int kp = k * p, R = p - 1, Cn = k - 1;
    const int npc = (Cn + GRAM_BLK - 1) / GRAM_BLK;
    double* tau = tau_all + (size_t)slot * kp;
    double* G = gram + (size_t)slot * (size_t)(R > 0 ? R : 1) * (Cn > 0 ? Cn : 1);
    const double* tr = traces + (size_t)slot * nmat;
    // Gram entries across the threads of a quarter block (neighbouring entries are neighbouring addresses), the CTA partials
    // split over the four quarters, combined in a fixed order
    __shared__ dd s_q[4][256];
    const int qtr = threadIdx.x >> 8, et = threadIdx.x & 255;
    for (int e0 = 0; e0 < R * Cn; e0 += 256) {
        const int e = e0 + et;
        dd s;
        s.hi = 0.0;
        s.lo = 0.0;
        if (e < R * Cn) {
            const int r = e / Cn, q = e - r * Cn;
            const int pass = (r / GRAM_BLK) * npc + q / GRAM_BLK;
            const double* src = partial + ((size_t)slot * npasses + pass) * nctas * (GRAM_BLK * GRAM_BLK) + (r % GRAM_BLK) * GRAM_BLK + q % GRAM_BLK;
            for (int cta = qtr; cta < nctas; cta += 4) s = dd_add_prod(s, __ldcs(src + (size_t)cta * (GRAM_BLK * GRAM_BLK)), 1.0);
        }
        s_q[qtr][et] = s;
        __syncthreads();
        if (qtr == 0 && e < R * Cn) {
            dd v = s_q[0][et];
            for (int g = 1; g < 4; ++g) v = dd_add(v, s_q[g][et]);
            G[e] = v.hi + v.lo;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) tau[0] = (double)N;
    for (int n = 1 + threadIdx.x; n <= k && n < kp; n += blockDim.x) tau[n] = tr[n - 1];
    __syncthreads();
    for (int j = 1; j < p; ++j) {
        if (threadIdx.x == 0 && j >= 2) tau[j * k] = tr[k + j - 2];  // tr U_j (tau_k = tr T_k is already set)
        for (int i = 1 + threadIdx.x; i < k; i += blockDim.x) tau[j * k + i] = 2.0 * G[(size_t)(j - 1) * Cn + (i - 1)] - tau[j * k - i];
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------------
// a-7: mu search.  N_e(mu) = sum_n c_n(mu) tau_n = sum_j f~(x_j; mu) w_j with the mu-independent weights
//   w_j = (1/N_q) sum_{n<M} (2 - delta_n0) tau_n cos(n theta_j)
// (the DCT of cheb_dm_coeffs with the two sums exchanged), so one bisection step costs N_q Fermi values.
//   mu_weights_kernel: block (j, slot) -> w[slot][j]
//   mu_bisect_kernel : one block per slot, `iters` halvings of [a,b]: N_e(mid) < n_occ ? lo = mid : hi = mid.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) mu_weights_kernel(const double* __restrict__ tau_all, const double* __restrict__ costab, int Nq, int M,
                                                         int kp, double* __restrict__ w_all) {
    __shared__ dd s_buf[32];
    const int j = blockIdx.x, slot = blockIdx.y;
    const double* tau = tau_all + (size_t)slot * kp;
    const unsigned mask = 4u * (unsigned)Nq - 1u;
    dd s;
    s.hi = 0.0;
    s.lo = 0.0;
    for (int n = threadIdx.x; n < M; n += blockDim.x) {
        const unsigned r = ((unsigned)n * (2u * (unsigned)j + 1u)) & mask;
        s = dd_add_prod(s, (n == 0 ? 1.0 : 2.0) * tau[n], costab[r]);
    }
    s = dd_block_reduce(s, s_buf);
    if (threadIdx.x == 0) w_all[(size_t)slot * Nq + j] = (s.hi + s.lo) / (double)Nq;
}

struct BisectArgs {
    double n_occ[MAX_BATCH];
};
// Fermi function for the electron count of the bisection only: beyond |y| = 44 it is 0 or 1 to 8e-20, which changes
// N_e = sum_j f_j w_j by less than 1e-14 (the coefficient tables keep the exact fermi_scaled); with beta~ of several
// hundred only a few per cent of the N_q nodes then pay for an exp, and neighbouring nodes share a warp.
__device__ __forceinline__ double fermi_count(double beta_t, double mu_t, double x) {
    const double y = beta_t * (x - mu_t);
    if (y > 44.0) return 0.0;
    if (y < -44.0) return 1.0;
    if (y > 0.0) {
        const double e = exp(-y);
        return e / (1.0 + e);
    }
    return 1.0 / (1.0 + exp(y));
}

// Three halvings per pass: the midpoints a bisection can visit in its next three steps form a binary tree of 7 points
// (node 1 = mid(lo, hi); node 2c, 2c+1 = the midpoints of the two halves of node c's interval, computed with the same
// expression 0.5 (lo + hi) the sequential bisection would use), N_e is evaluated at all 7 in one pass over the nodes and
// one block reduction, and thread 0 then walks the tree with the sequential rule.  The result is bit-identical to one
// halving per pass; the passes (block reduction latency, not the N_q Fermi values) drop from 101 to 35.
constexpr int BISECT_LEVELS = 3, BISECT_POINTS = (1 << BISECT_LEVELS) - 1;
// Work split of a pass: thread t evaluates point c = t % 8 (the eighth is idle) at the nodes j = t / 8, t / 8 + 64, ...:
// the few nodes near mu that need an exp (an FP64 exp is ~1000 cycles of dependent instructions) are neighbours, so they
// land on different threads and a pass costs one exp latency, not 7 x (nodes per thread) of them.
__global__ void __launch_bounds__(512) mu_bisect_kernel(DevScalars* sc_all, double beta, const BisectArgs B, int iters,
                                                        const double* __restrict__ costab, int Nq, const double* __restrict__ w_all) {
    __shared__ dd s_part[8][16];
    __shared__ double s_nepts[8];
    __shared__ double s_lo, s_hi, s_ne;
    __shared__ int s_fixed;  // a pass left [lo, hi] unchanged: every further halving is a no-op
    DevScalars* sc = sc_all + blockIdx.x;
    const double* w = w_all + (size_t)blockIdx.x * Nq;
    const double n_occ = B.n_occ[blockIdx.x];
    const double a = sc->a, b = sc->b;
    const double beta_t = beta * (b - a) * 0.5;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int c = threadIdx.x & 7, grp = threadIdx.x >> 3, ngrp = blockDim.x >> 3;
    if (threadIdx.x == 0) { s_lo = a; s_hi = b; s_ne = 0.0; s_fixed = 0; }
    __syncthreads();
    int done = 0;
    while (done <= iters) {
        // levels of this pass: up to 3 halvings; the last pass evaluates N_e at the returned mu only (one point)
        const int levels = (done == iters) ? 1 : min(BISECT_LEVELS, iters - done);
        const int npts = (1 << levels) - 1;
        double lo_[BISECT_POINTS + 1], hi_[BISECT_POINTS + 1], mid[BISECT_POINTS + 1];
        lo_[1] = s_lo;
        hi_[1] = s_hi;
#pragma unroll
        for (int q = 1; q <= BISECT_POINTS; ++q) {
            mid[q] = 0.5 * (lo_[q] + hi_[q]);
            if (2 * q + 1 <= BISECT_POINTS) {
                lo_[2 * q] = lo_[q];       hi_[2 * q] = mid[q];       // N_e(mid) >= n_occ: hi = mid
                lo_[2 * q + 1] = mid[q];   hi_[2 * q + 1] = hi_[q];   // N_e(mid) <  n_occ: lo = mid
            }
        }
        double my_mid = 0.0;
#pragma unroll
        for (int q = 1; q <= BISECT_POINTS; ++q)
            if (q == c + 1) my_mid = mid[q];
        const double mu_t = (2.0 * my_mid - (a + b)) / (b - a);
        dd s, s1;  // two independent accumulation chains (a double-double step is ~100 cycles of dependent instructions)
        s.hi = s.lo = s1.hi = s1.lo = 0.0;
        if (c < npts) {
            int j = grp;
            for (; j + ngrp < Nq; j += 2 * ngrp) {
                s = dd_add_prod(s, fermi_count(beta_t, mu_t, costab[2 * j + 1]), w[j]);
                s1 = dd_add_prod(s1, fermi_count(beta_t, mu_t, costab[2 * (j + ngrp) + 1]), w[j + ngrp]);
            }
            if (j < Nq) s = dd_add_prod(s, fermi_count(beta_t, mu_t, costab[2 * j + 1]), w[j]);
            s = dd_add(s, s1);
        }
        // fixed-order reduction per point: the 4 lanes of a warp with the same c, then the warps
#pragma unroll
        for (int o = 16; o >= 8; o >>= 1) {
            dd other;
            other.hi = __shfl_down_sync(0xffffffffu, s.hi, o);
            other.lo = __shfl_down_sync(0xffffffffu, s.lo, o);
            s = dd_add(s, other);
        }
        if (lane < 8) s_part[lane][warp] = s;
        __syncthreads();
        if (warp == 0) {
            {   // lane (qq, c): warps 4 qq .. 4 qq + 3 of point c, then the four quarters (fixed order)
                const int qq = lane >> 3;
                dd v;
                v.hi = v.lo = 0.0;
                for (int q = 4 * qq; q < 4 * qq + 4 && q < nw; ++q) v = dd_add(v, s_part[c][q]);
#pragma unroll
                for (int o = 16; o >= 8; o >>= 1) {
                    dd other;
                    other.hi = __shfl_down_sync(0xffffffffu, v.hi, o);
                    other.lo = __shfl_down_sync(0xffffffffu, v.lo, o);
                    v = dd_add(v, other);
                }
                if (lane < 8) s_nepts[lane] = v.hi + v.lo;
            }
            __syncwarp();
            if (lane == 0) {
                if (done == iters) {
                    s_ne = s_nepts[0];  // N_e at the returned mu = (lo + hi) / 2
                } else {
                    int q = 1;
                    double lo = lo_[1], hi = hi_[1];
                    for (int l = 0; l < levels; ++l) {
                        double m_q = 0.0;   // select without dynamic indexing of the register array
#pragma unroll
                        for (int r = 1; r <= BISECT_POINTS; ++r)
                            if (r == q) m_q = mid[r];
                        if (s_nepts[q - 1] < n_occ) { lo = m_q; q = 2 * q + 1; } else { hi = m_q; q = 2 * q; }
                    }
                    // (the interval reaches the spacing of the doubles after ~60 halvings; the state is a function of
                    // (lo, hi) alone, so once a pass does not move it the remaining halvings would not either)
                    if (lo == lo_[1] && hi == hi_[1]) s_fixed = 1;
                    s_lo = lo;
                    s_hi = hi;
                }
            }
        }
        __syncthreads();
        if (done == iters) done += 1;
        else if (s_fixed) done = iters;  // skip the no-op halvings; the result is bitwise that of `iters` halvings
        else done += levels;
    }
    if (threadIdx.x == 0) {
        sc->mu = 0.5 * (s_lo + s_hi);
        sc->ne = s_ne;
    }
}

// ---------------------------------------------------------------------------------------------------
// a-5, batched form (SURVEY 8(a) option ii; Eq. 21): all low-order sums at once,
//     G_l = coefT[l][0] I + sum_{i=1}^{k-1} coefT[l][i] T_i,   l < p   (coefT = g or d, layout [l*k + i]),
// reading every T_i once per chunk of SUMS_CHUNK outputs instead of once per giant step: HBM bytes
// (ceil(p/SUMS_CHUNK) (k-1) + p) mat instead of p (k-1) mat for the epilogue-fused form.  One thread owns
// one 16-byte element pair of the padded matrices (pad columns are zero in every T_i, so they stay zero).
//   grid = (ceil(pairs / 256), ceil(p / SUMS_CHUNK)), block = 256.
// ---------------------------------------------------------------------------------------------------
constexpr int SUMS_CHUNK = 16;
// With symmetric-tile skipping (symBM > 0) only the elements inside tiles that are work items of the giant steps are
// formed (tile (tm, tn) of symBM x symBN with tm symBM + symBM - 1 >= tn symBN): the other tiles of G_l are never read.
__global__ void __launch_bounds__(256) form_sums_kernel(const double* __restrict__ Tbase0, long long stride, long long ld, int N, int k,
                                                        int p, const double* __restrict__ coefT0, double* __restrict__ Gbase0,
                                                        int symBM, int symBN, long long slot_stride) {
    extern __shared__ double s_coef[];  // [k][SUMS_CHUNK]
    const double* __restrict__ Tbase = Tbase0 + (long long)blockIdx.z * slot_stride;   // blockIdx.z = matrix of the batch
    double* __restrict__ Gbase = Gbase0 + (long long)blockIdx.z * slot_stride;
    const double* __restrict__ coefT = coefT0 + (size_t)blockIdx.z * k * p;
    const int l0 = blockIdx.y * SUMS_CHUNK;
    const int nl = min(SUMS_CHUNK, p - l0);
    for (int e = threadIdx.x; e < k * SUMS_CHUNK; e += blockDim.x) {
        const int i = e / SUMS_CHUNK, q = e - i * SUMS_CHUNK;
        s_coef[e] = (q < nl) ? coefT[(size_t)(l0 + q) * k + i] : 0.0;
    }
    __syncthreads();
    const long long pairs = (long long)N * ld / 2;
    const long long pr = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (pr >= pairs) return;
    const long long e0 = 2 * pr;
    const int row = (int)(e0 / ld), col = (int)(e0 - (long long)row * ld);
    if (symBM > 0 && (row / symBM) * symBM + symBM - 1 < (col / symBN) * symBN) return;  // tile not needed
    double2 acc[SUMS_CHUNK];
#pragma unroll
    for (int q = 0; q < SUMS_CHUNK; ++q) acc[q] = make_double2(0.0, 0.0);
    const double* src = Tbase + e0;
    int i = 1;
    for (; i + 3 < k; i += 4) {
        double2 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = __ldcs(reinterpret_cast<const double2*>(src + (long long)(i - 1 + u) * stride));
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int q = 0; q < SUMS_CHUNK; ++q) {
                const double w = s_coef[(i + u) * SUMS_CHUNK + q];
                acc[q].x = fma(w, v[u].x, acc[q].x);
                acc[q].y = fma(w, v[u].y, acc[q].y);
            }
    }
    for (; i < k; ++i) {
        const double2 v = __ldcs(reinterpret_cast<const double2*>(src + (long long)(i - 1) * stride));
#pragma unroll
        for (int q = 0; q < SUMS_CHUNK; ++q) {
            const double w = s_coef[i * SUMS_CHUNK + q];
            acc[q].x = fma(w, v.x, acc[q].x);
            acc[q].y = fma(w, v.y, acc[q].y);
        }
    }
    const bool d0 = (col == row), d1 = (col + 1 == row);
#pragma unroll
    for (int q = 0; q < SUMS_CHUNK; ++q) {
        if (q < nl) {
            double2 o = acc[q];
            if (d0) o.x += s_coef[q];
            if (d1) o.y += s_coef[q];
            *reinterpret_cast<double2*>(Gbase + (long long)(l0 + q) * stride + e0) = o;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// a-5, batched form on the tensor cores.  The batched sums are themselves a skinny GEMM,
//     G[e][l] = sum_i T_i[e] coefT[l][i]        (e = matrix element, K = k - 1, N = p),
// and the scalar kernel above is bound by the FP64 FMA pipe (2 N^2 (k-1) p flops at 64 FMA/clk/SM: 1.0 ms at cfg4),
// not by HBM.  Here one warp owns 32 consecutive elements (4 m-blocks of 8) x SUMS_CHUNK sums (2 n-blocks of 8):
// per k4-step 4 scalar loads per lane (lane (g, t) reads element g of matrix i0 + t: 64-byte segments), 2 coefficient
// fragments from shared memory and 8 DMMA.8x8x4.  Same skipping of unneeded tiles, same diagonal term.
//   grid = (ceil(N ld / 32 / 8), ceil(p / SUMS_CHUNK)), block = 256 (8 warps).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) form_sums_dmma_kernel(const double* __restrict__ Tbase0, long long stride, long long ld, int N, int k,
                                                             int p, const double* __restrict__ coefT0, double* __restrict__ Gbase0,
                                                             int symBM, int symBN, long long slot_stride) {
    extern __shared__ double s_coef[];  // [kpad][SUMS_CHUNK], kpad = (k - 1) rounded up to 4; row i - 1 <-> T_i; + [SUMS_CHUNK] diag
    const double* __restrict__ Tbase = Tbase0 + (long long)blockIdx.z * slot_stride;   // blockIdx.z = matrix of the batch
    double* __restrict__ Gbase = Gbase0 + (long long)blockIdx.z * slot_stride;
    const double* __restrict__ coefT = coefT0 + (size_t)blockIdx.z * k * p;
    const int l0 = blockIdx.y * SUMS_CHUNK;
    const int nl = min(SUMS_CHUNK, p - l0);
    const int kk = k - 1, kpad = (kk + 3) & ~3;
    for (int e = threadIdx.x; e < (kpad + 1) * SUMS_CHUNK; e += blockDim.x) {
        const int i = e / SUMS_CHUNK, q = e - i * SUMS_CHUNK;  // i == kpad: coefficient of T_0 = I
        const int src_i = (i == kpad) ? 0 : i + 1;
        s_coef[e] = (q < nl && (i == kpad || i < kk)) ? coefT[(size_t)(l0 + q) * k + src_i] : 0.0;
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, t = lane & 3;
    const long long total = (long long)N * ld;
    const long long e0 = ((long long)blockIdx.x * 8 + warp) * 32;
    if (e0 >= total) return;
    bool need[4];
    bool any = false;
#pragma unroll
    for (int mb = 0; mb < 4; ++mb) {
        const long long e = e0 + mb * 8;  // an 8-block never crosses a row (ld is a multiple of 16) nor a tile
        const int row = (int)(e / ld), col = (int)(e - (long long)row * ld);
        need[mb] = (e < total) && !(symBM > 0 && (row / symBM) * symBM + symBM - 1 < (col / symBN) * symBN);
        any = any || need[mb];
    }
    if (!any) return;
    double acc[4][2][2];
#pragma unroll
    for (int mb = 0; mb < 4; ++mb)
#pragma unroll
        for (int nb = 0; nb < 2; ++nb) acc[mb][nb][0] = acc[mb][nb][1] = 0.0;
    const double* src = Tbase + e0 + g;
    for (int i0 = 0; i0 < kpad; i0 += 4) {
        const int it = min(i0 + t, kk - 1);  // padded k-rows carry a zero coefficient; read a valid matrix
        const double* ps = src + (long long)it * stride;
        double a[4], b[2];
#pragma unroll
        for (int mb = 0; mb < 4; ++mb) a[mb] = need[mb] ? __ldcs(ps + mb * 8) : 0.0;
#pragma unroll
        for (int nb = 0; nb < 2; ++nb) b[nb] = s_coef[(i0 + t) * SUMS_CHUNK + nb * 8 + g];
#pragma unroll
        for (int mb = 0; mb < 4; ++mb)
#pragma unroll
            for (int nb = 0; nb < 2; ++nb) dmma_884(acc[mb][nb][0], acc[mb][nb][1], a[mb], b[nb]);
    }
#pragma unroll
    for (int mb = 0; mb < 4; ++mb) {
        if (!need[mb]) continue;
        const long long e = e0 + mb * 8 + g;
        const int row = (int)(e / ld), col = (int)(e - (long long)row * ld);
#pragma unroll
        for (int nb = 0; nb < 2; ++nb)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int q = nb * 8 + 2 * t + h;
                if (q < nl) {
                    double v = acc[mb][nb][h];
                    if (row == col) v += s_coef[kpad * SUMS_CHUNK + q];
                    Gbase[(long long)(l0 + q) * stride + e] = v;
                }
            }
    }
}

// ---------------------------------------------------------------------------------------------------
// Roofline denominator: register-resident DMMA.8x8x4 issue-rate microbenchmark (cheb_dm_dmma_peak).
// Each warp runs DMMA_PEAK_CHAINS independent accumulator chains; no memory traffic in the loop.
// ---------------------------------------------------------------------------------------------------
constexpr int DMMA_PEAK_CHAINS = 8;
__global__ void __launch_bounds__(512) dmma_peak_kernel(int iters, double* sink) {
    double c[DMMA_PEAK_CHAINS][2];
#pragma unroll
    for (int i = 0; i < DMMA_PEAK_CHAINS; ++i) c[i][0] = c[i][1] = 0.0;
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < DMMA_PEAK_CHAINS; ++i) dmma_884(c[i][0], c[i][1], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < DMMA_PEAK_CHAINS; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) sink[threadIdx.x & 63] = s;  // keeps the chains alive
}

}  // namespace chebdm
