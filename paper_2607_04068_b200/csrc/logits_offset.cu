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
// The caller clamps the logit to (max - 700) in fp32 first (one FMNMX; a double fmax costs five instructions):
// terms that small cannot move a sum that is >= 1, and -inf logits never reach the fp64 code.
// The full-width fp64 constants live in constant memory and are used as constant-bank operands: written as
// literals, ptxas rebuilt each of them with two MOVs per use (47 instructions per element, issue-bound).
__constant__ double kExpC[6] = {92.332482616893656,       // 64 / ln2
                                -0.01083042469326756,      // -(ln2/64), high part: 32 significant bits
                                -2.9815858269852933e-12,   // -(ln2/64), low part
                                1.0 / 120.0, 1.0 / 24.0, 1.0 / 6.0};

__device__ __forceinline__ double exp_neg(double d, const double* __restrict__ tab) {
    const double kMagic = 6755399441055744.0;                 // 2^52 + 2^51: round-to-nearest-integer by addition
    const double t = fma(d, kExpC[0], kMagic);
    const int k = __double2loint(t);                          // integer in the low word (two's complement)
    const double kf = t - kMagic;
    // r = d - k ln2/64 in two steps: kf * high part is exact for |k| < 2^20
    double r = fma(kf, kExpC[1], d);
    r = fma(kf, kExpC[2], r);
    double p = fma(r, kExpC[3], kExpC[4]);
    p = fma(p, r, kExpC[5]);
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

    const long long stride = (long long)gridDim.x * kRows;
    auto finish = [&](long long row, bool live, float m, double s) {
        s = row_sum<kTPR>(s, sd);
        if (live && t == 0) {
            float o = ninf;  // a beam without a legal continuation
            if (m != ninf) {
                const float lse = __double2float_rn((double)m + log(s));
                o = __fsub_rn(score ? __ldg(score + row) : 0.f, lse);
            }
            offset[row] = o;
        }
    };

    if (vec) {
        // One row at a time per CTA, 64 registers, 4 CTAs per SM.  Measured at C = 8192 (B200, 134 MB): a register
        // double buffer that requests the next row before this row's arithmetic needs 128 registers (2 CTAs per
        // SM) and is slower (52.7 us against 49.6 us): the kernel is bound by fp64 issue, not by load latency.
        const int C4 = C >> 2;
        float4 nx[kRegVec];
        auto load_row = [&](long long r0) {
            const long long row = r0 + r_in;
            const float4* __restrict__ p4 = reinterpret_cast<const float4*>(logits + (row < rows ? row : 0) * (long long)C);
#pragma unroll
            for (int x = 0; x < kRegVec; ++x) {
                const int j = x * kTPR + t;
                nx[x] = make_float4(ninf, ninf, ninf, ninf);
                if (row < rows && j < C4) nx[x] = __ldg(p4 + j);
            }
        };
        long long row0 = (long long)blockIdx.x * kRows;
        for (; row0 < rows; row0 += stride) {
            load_row(row0);
            const long long row = row0 + r_in;
            const bool live = row < rows;  // uniform per warp (kTPR >= 32)
            const float4* __restrict__ p4 = reinterpret_cast<const float4*>(logits + (live ? row : 0) * (long long)C);
            float4 v[kRegVec];
#pragma unroll
            for (int x = 0; x < kRegVec; ++x) v[x] = nx[x];
            float m = ninf;
#pragma unroll
            for (int x = 0; x < kRegVec; ++x) m = fmaxf(m, max4(v[x]));
            if (live)
                for (int j = kRegVec * kTPR + t; j < C4; j += kTPR) m = fmaxf(m, max4(__ldg(p4 + j)));
            m = row_max<kTPR>(m, sm);
            double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
            if (m != ninf) {  // uniform per row
                const double md = (double)m;
                const float mlo = m - 700.f;
#pragma unroll
                for (int x = 0; x < kRegVec; ++x) {
                    if (x * kTPR + t < C4) {
                        s0 += exp_neg((double)fmaxf(v[x].x, mlo) - md, tab); s1 += exp_neg((double)fmaxf(v[x].y, mlo) - md, tab);
                        s2 += exp_neg((double)fmaxf(v[x].z, mlo) - md, tab); s3 += exp_neg((double)fmaxf(v[x].w, mlo) - md, tab);
                    }
                }
                for (int j = kRegVec * kTPR + t; j < C4; j += kTPR) {
                    const float4 w = __ldg(p4 + j);
                    s0 += exp_neg((double)fmaxf(w.x, mlo) - md, tab); s1 += exp_neg((double)fmaxf(w.y, mlo) - md, tab);
                    s2 += exp_neg((double)fmaxf(w.z, mlo) - md, tab); s3 += exp_neg((double)fmaxf(w.w, mlo) - md, tab);
                }
            }
            finish(row, live, m, (s0 + s1) + (s2 + s3));
        }
        return;
    }

    for (long long row0 = (long long)blockIdx.x * kRows; row0 < rows; row0 += stride) {
        const long long row = row0 + r_in;
        const bool live = row < rows;
        const float* __restrict__ p = logits + (live ? row : 0) * (long long)C;
        float m = ninf;
        double s = 0.0;
        {
            if (live)
                for (int j = t; j < C; j += kTPR) m = fmaxf(m, __ldg(p + j));
            m = row_max<kTPR>(m, sm);
            if (m != ninf) {
                const double md = (double)m;
                const float mlo = m - 700.f;
                for (int j = t; j < C; j += kTPR) s += exp_neg((double)fmaxf(__ldg(p + j), mlo) - md, tab);
            }
        }
        finish(row, live, m, s);
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
