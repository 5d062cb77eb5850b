// Selection straight from raw logits (reading R22).
//
// Eq. 1 scores a path by the sum of log P(c_j | ...) = logit - logsumexp(logits of the
// parent beam).  The normaliser is ONE scalar per parent beam, so it is folded into the beam's running score
// and the candidates are never rewritten:
//     lse[i]    = fl32( logsumexp_c logits[i, c] )     fp64 arithmetic, rounded once
//     offset[i] = fl32( score[i] - lse[i] )            one fp32 subtraction; all logits -inf => -inf
//     key[i*C + c] = fl32( offset[i] + logits[i, c] )  the A3 kernels, fed (logits, offset)
// A log-softmax kernel in front of A3 would read the logits, write C log-probs per beam and A3 would read them
// again (12 B per candidate); this path reads the logits here and in A3 (8 B per candidate, the second read
// mostly from L2 at the benchmark sizes) and writes 4 B per BEAM.
//
// HBM-bound stream: 4 B per candidate read once; the row stays in registers between the max pass and the
// sum pass (up to 32 floats per thread; longer rows re-read their tail through L1/L2).  A warp per row for
// C <= 1024, a 256-thread CTA per row above.  The exponentials are fp64 (exp_neg below) so that the fp32
// result is the correctly rounded one the oracle defines (a different summation order or a last-bit
// difference of exp moves the fp64 sum by ~1e-16 relative: a flipped fp32 rounding needs the exact value
// within ~1e-9 ulp of a rounding boundary).
#include <math.h>

#include "common.cuh"

namespace stark {

namespace {

constexpr int kThreads = 256;
constexpr int kRegVec = 8;  // float4 per thread kept between the two passes

// exp(d) for d <= 0 in fp64, error < 1 ulp + the table's: d = (64 e + j) ln2/64 + r, |r| <= ln2/128,
// exp(d) = 2^e * 2^(j/64) * exp(r).  exp(r) is the degree-5 Taylor polynomial (remainder r^6/720 < 3.6e-17);
// 2^(j/64) comes from a 64-entry shared-memory table (filled with exp2() by each CTA); 2^e is an exponent
// add.  13 fp64 operations against ~25 of the library exp(): the kernel is fp64-pipe-bound at large C.
// Terms below e^-700 (they cannot move a sum that is >= 1) return 0, which also covers d = -inf.
__device__ __forceinline__ double exp_neg(double d, const double* __restrict__ tab) {
    if (d < -700.0) return 0.0;
    const double kMagic = 6755399441055744.0;                 // 2^52 + 2^51: round-to-nearest-integer by addition
    const double t = fma(d, 92.332482616893656, kMagic);      // d * 64/ln2
    const int k = __double2loint(t);                          // integer in the low word (two's complement)
    const double kf = t - kMagic;
    // r = d - k ln2/64 in two steps: the high part has 32 significant bits, so kf * hi is exact for |k| < 2^20
    double r = fma(kf, -0.01083042469326756, d);
    r = fma(kf, -2.9815858269852933e-12, r);
    double p = fma(r, 1.0 / 120.0, 1.0 / 24.0);
    p = fma(p, r, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    const double v = tab[k & 63] * p;                          // in (0.99, 2.01)
    const int e = k >> 6;                                      // floor(k / 64) >= -1010: the result stays normal
    return __hiloint2double(__double2hiint(v) + (e << 20), __double2loint(v));
}

__device__ __forceinline__ float max4(float4 v) { return fmaxf(fmaxf(v.x, v.y), fmaxf(v.z, v.w)); }

template <int kTPR>  // threads per row: 32 (warp) or 256 (CTA)
__device__ __forceinline__ float row_max(float m, float* sm) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    if constexpr (kTPR > 32) {
        const int warp = threadIdx.x >> 5;
        __syncthreads();  // sm free again
        if ((threadIdx.x & 31) == 0) sm[warp] = m;
        __syncthreads();
        m = sm[0];
#pragma unroll
        for (int w = 1; w < kTPR / 32; ++w) m = fmaxf(m, sm[w]);
    }
    return m;
}

template <int kTPR>
__device__ __forceinline__ double row_sum(double s, double* sd) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if constexpr (kTPR > 32) {
        const int warp = threadIdx.x >> 5;
        __syncthreads();
        if ((threadIdx.x & 31) == 0) sd[warp] = s;
        __syncthreads();
        s = sd[0];
#pragma unroll
        for (int w = 1; w < kTPR / 32; ++w) s += sd[w];
    }
    return s;
}

template <int kTPR>
__global__ void __launch_bounds__(kThreads)
row_offset_kernel(const float* __restrict__ logits, const float* __restrict__ score, long long rows, int C,
                  int vec, float* __restrict__ offset) {
    constexpr int kRows = kThreads / kTPR;  // rows per CTA and iteration
    __shared__ float sm[kThreads / 32];
    __shared__ double sd[kThreads / 32];
    __shared__ double tab[64];  // 2^(j/64)
    if (threadIdx.x < 64) tab[threadIdx.x] = exp2((double)threadIdx.x * (1.0 / 64.0));
    __syncthreads();
    const int t = threadIdx.x % kTPR, r_in = threadIdx.x / kTPR;
    const float ninf = __int_as_float(0xff800000);

    for (long long row0 = (long long)blockIdx.x * kRows; row0 < rows; row0 += (long long)gridDim.x * kRows) {
        const long long row = row0 + r_in;
        const bool live = row < rows;  // uniform per warp (kTPR >= 32)
        const float* __restrict__ p = logits + (live ? row : 0) * (long long)C;
        float m = ninf;
        double s = 0.0;
        if (vec) {
            const float4* __restrict__ p4 = reinterpret_cast<const float4*>(p);
            const int C4 = C >> 2;
            float4 v[kRegVec];
#pragma unroll
            for (int x = 0; x < kRegVec; ++x) {
                const int j = x * kTPR + t;
                v[x] = make_float4(ninf, ninf, ninf, ninf);
                if (live && j < C4) v[x] = __ldg(p4 + j);
            }
#pragma unroll
            for (int x = 0; x < kRegVec; ++x) m = fmaxf(m, max4(v[x]));
            if (live)
                for (int j = kRegVec * kTPR + t; j < C4; j += kTPR) m = fmaxf(m, max4(__ldg(p4 + j)));
            m = row_max<kTPR>(m, sm);
            if (m != ninf) {  // uniform per row
                const double md = (double)m;
#pragma unroll
                for (int x = 0; x < kRegVec; ++x) {
                    if (x * kTPR + t < C4) {
                        s += exp_neg((double)v[x].x - md, tab); s += exp_neg((double)v[x].y - md, tab);
                        s += exp_neg((double)v[x].z - md, tab); s += exp_neg((double)v[x].w - md, tab);
                    }
                }
                for (int j = kRegVec * kTPR + t; j < C4; j += kTPR) {
                    const float4 w = __ldg(p4 + j);
                    s += exp_neg((double)w.x - md, tab); s += exp_neg((double)w.y - md, tab);
                    s += exp_neg((double)w.z - md, tab); s += exp_neg((double)w.w - md, tab);
                }
            }
        } else {
            if (live)
                for (int j = t; j < C; j += kTPR) m = fmaxf(m, __ldg(p + j));
            m = row_max<kTPR>(m, sm);
            if (m != ninf) {
                const double md = (double)m;
                for (int j = t; j < C; j += kTPR) s += exp_neg((double)__ldg(p + j) - md, tab);
            }
        }
        s = row_sum<kTPR>(s, sd);
        if (live && t == 0) {
            float o = ninf;  // a beam without a legal continuation
            if (m != ninf) {
                const float lse = __double2float_rn((double)m + log(s));
                o = __fsub_rn(score ? __ldg(score + row) : 0.f, lse);
            }
            offset[row] = o;
        }
    }
}

}  // namespace

int launch_row_offset(const float* logits, const float* score, long long rows, int C, float* offset,
                      cudaStream_t st) {
    const int vec = (C & 3) == 0 && (reinterpret_cast<uintptr_t>(logits) & 15u) == 0;
    if (C <= 1024) {
        long long nb = (rows + 7) / 8;
        if (nb > 148 * 16) nb = 148 * 16;
        row_offset_kernel<32><<<(unsigned)nb, kThreads, 0, st>>>(logits, score, rows, C, vec, offset);
    } else {
        long long nb = rows;
        if (nb > 148 * 8) nb = 148 * 8;
        row_offset_kernel<256><<<(unsigned)nb, kThreads, 0, st>>>(logits, score, rows, C, vec, offset);
    }
    STARK_LAUNCH_CHECK();
    return STARK_OK;
}

}  // namespace stark
