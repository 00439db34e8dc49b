// fft.cuh -- the Fourier transform of SURVEY.md 8(f)-1 (step iv of P:408), hand-written: batched complex DFTs of ANY
// length n in fp64 on the device.
//
//   n a power of two : Stockham autosort passes of radix 16 (then 4 / 2 for the remaining bits), every pass one read and
//                      one write of the series (HBM-bound: 32 B per point and pass); the radix-16 butterfly runs in
//                      registers as 4 x 4 with the W16 twiddles between the two layers.
//   any other n      : Bluestein's chirp-z identity  j k = (j^2 + k^2 - (k - j)^2) / 2 :
//                        Z_k = c_k sum_j (z_j c_j) conj(c)_{k-j},   c_j = exp(-i pi j^2 / n),
//                      a circular convolution of length m = 2^p >= 2 n - 1, done with the power-of-two transform: pack
//                      z c into m points, forward FFT, multiply by the transform of the wrapped conj(c), inverse FFT; the
//                      final c_k (and 1 / m) is applied where the spectrum is consumed.  j^2 mod 2 n is formed in 64-bit
//                      integers, so the chirp phases are exact multiples of pi / n before sincospi.
// Two real series ride in one complex transform (z = a + i b): a~_k = (Z_k + conj Z_{n-k}) / 2,
// b~_k = (Z_k - conj Z_{n-k}) / (2 i): the six real transforms of a source pair (A, E, T of two responses) are three
// complex ones.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define FFT_THREADS 256

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x)); }
__device__ __forceinline__ double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
/* multiply by -i (SIGN = -1: forward) or +i (SIGN = +1) */
template <int SIGN>
__device__ __forceinline__ double2 cmul_i(double2 a) { return SIGN < 0 ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x); }

/* in-place DFT of 4 points with stride S in a register array: X_k = sum_n x_n exp(SIGN 2 pi i n k / 4) */
template <int SIGN, int S>
__device__ __forceinline__ void dft4(double2 *v)
{
    const double2 s02 = cadd(v[0], v[2 * S]), d02 = csub(v[0], v[2 * S]);
    const double2 s13 = cadd(v[S], v[3 * S]), d13 = cmul_i<SIGN>(csub(v[S], v[3 * S]));
    v[0] = cadd(s02, s13);
    v[S] = cadd(d02, d13);
    v[2 * S] = csub(s02, s13);
    v[3 * S] = csub(d02, d13);
}

/* DFT of R = 2, 4, 16 points in registers, natural order in and out */
template <int R, int SIGN>
__device__ __forceinline__ void dft_small(double2 *v)
{
    if (R == 2) {
        const double2 a = v[0], b = v[1];
        v[0] = cadd(a, b);
        v[1] = csub(a, b);
    } else if (R == 4) {
        dft4<SIGN, 1>(v);
    } else {
        /* n = 4 n1 + n2, k = k1 + 4 k2: DFT4 over n1 (stride 4) for every n2, twiddle W16^(n2 k1), DFT4 over n2 */
#pragma unroll
        for (int n2 = 0; n2 < 4; ++n2) dft4<SIGN, 4>(v + n2);   /* v[4 k1 + n2] */
        const double c1 = 0.92387953251128675613, s1 = 0.38268343236508977173, h = 0.70710678118654752440;
        const double sg = SIGN < 0 ? -1.0 : 1.0;
        const double2 w1 = make_double2(c1, sg * s1), w2 = make_double2(h, sg * h), w3 = make_double2(s1, sg * c1);
        const double2 w6 = make_double2(-h, sg * h), w9 = make_double2(-c1, -sg * s1);
        v[4 * 1 + 1] = cmul(v[4 * 1 + 1], w1); v[4 * 1 + 2] = cmul(v[4 * 1 + 2], w2); v[4 * 1 + 3] = cmul(v[4 * 1 + 3], w3);
        v[4 * 2 + 1] = cmul(v[4 * 2 + 1], w2); v[4 * 2 + 2] = cmul_i<SIGN>(v[4 * 2 + 2]); v[4 * 2 + 3] = cmul(v[4 * 2 + 3], w6);
        v[4 * 3 + 1] = cmul(v[4 * 3 + 1], w3); v[4 * 3 + 2] = cmul(v[4 * 3 + 2], w6); v[4 * 3 + 3] = cmul(v[4 * 3 + 3], w9);
        double2 o[16];
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) {
            dft4<SIGN, 1>(v + 4 * k1);                       /* over n2: v[4 k1 + k2] */
#pragma unroll
            for (int k2 = 0; k2 < 4; ++k2) o[k1 + 4 * k2] = v[4 * k1 + k2];
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = o[i];
    }
}

/* Where the first pass of a transform takes its input from: a complex buffer, or -- fused packing -- two real series
 * per complex series (z = a + i b, times the Bluestein chirp if C is given, zero beyond n) */
struct FftSource {
    const double2 *in;          /* complex input (series q at q * stride), or nullptr: pack from the real series below */
    const double *xa[3], *xb[3];
    int64_t ld, n;
    const double2 *C;
};
template <bool PACK>
__device__ __forceinline__ double2 fft_load(const FftSource &src, int64_t q, int64_t stride, int64_t j)
{
    if (!PACK) return src.in[q * stride + j];
    /* branch-free loads (clamped index, selected afterwards): the sixteen loads of a thread stay in flight together */
    const int64_t s = q / 3;
    const int c = (int)(q - 3 * s);
    const int64_t jc = j < src.n ? j : src.n - 1;
    double2 z = make_double2(src.xa[c][s * src.ld + jc], src.xb[c][s * src.ld + jc]);
    if (src.C) z = cmul(z, src.C[jc]);
    return j < src.n ? z : make_double2(0.0, 0.0);
}

/* One Stockham pass of radix R over series of N points (grid.y = series): thread j < N / R reads x[j + r N / R], applies
 * the twiddles exp(SIGN 2 pi i r (j mod Ns) / (Ns R)), transforms R points and writes them Ns apart.  After the passes
 * with Ns = 1, R1, R1 R2, ... the series is transformed in natural order (autosort: no bit reversal). */
template <int R, int SIGN, bool PACK>
__global__ void __launch_bounds__(FFT_THREADS) fft_pass_kernel(const __grid_constant__ FftSource src, double2 *__restrict__ out, int N,
                                                               int Ns, int64_t stride)
{
    const int j = blockIdx.x * FFT_THREADS + threadIdx.x;
    const int T = N / R;
    if (j >= T) return;
    out += (int64_t)blockIdx.y * stride;
    double2 v[R];
#pragma unroll
    for (int r = 0; r < R; ++r) v[r] = fft_load<PACK>(src, blockIdx.y, stride, (int64_t)j + (int64_t)r * T);
    const int k = j & (Ns - 1);
    if (Ns > 1) {
        /* w_r = exp(SIGN 2 pi i r k / (Ns R)): the powers of two by sincospi of an exact argument, the others as products */
        const double base = (double)k / (double)(Ns * (R / 2));     /* 2 k / (Ns R), exact */
        double2 wp[4];
#pragma unroll
        for (int b = 0; (1 << b) < R; ++b) {
            double s, c;
            sincospi(base * (double)(1 << b), &s, &c);
            wp[b] = make_double2(c, SIGN < 0 ? -s : s);
        }
#pragma unroll
        for (int r = 1; r < R; ++r) {
            double2 w = make_double2(1.0, 0.0);
            bool first = true;
#pragma unroll
            for (int b = 0; (1 << b) < R; ++b)
                if (r & (1 << b)) { w = first ? wp[b] : cmul(w, wp[b]); first = false; }
            v[r] = cmul(v[r], w);
        }
    }
    dft_small<R, SIGN>(v);
    const int j0 = (j / Ns) * Ns * R + k;
#pragma unroll
    for (int r = 0; r < R; ++r) out[j0 + r * Ns] = v[r];
}

/* exp(SIGN 2 pi i e / 256), e = 0 .. 255 (cos, -sin stored: SIGN = -1; the other sign by conjugation) */
__constant__ double2 c_w256[256];

/* One Stockham pass of radix 256 through shared memory: a block of 256 threads takes 16 consecutive j < N / 256 and their
 * 256 inputs x[j + r N / 256] each.  With r = c + 16 r1 and the output index q = q1 + 16 q2,
 *   X[q1 + 16 q2] = sum_c W16^(c q2) [ W256^(c q1) sum_r1 W16^(r1 q1) x[c + 16 r1] ] :
 * thread (jj, c) transforms the 16 inputs of residue c and applies W256^(c q1), the block transposes through shared
 * memory (rows padded to 17: conflict free both ways), thread (jj, q1) transforms over c and writes Ns apart.  One read
 * and one write of the series for eight bits of the length (two radix-16 passes would move it twice). */
template <int SIGN, bool PACK>
__global__ void __launch_bounds__(256) fft_pass256_kernel(const __grid_constant__ FftSource src, double2 *__restrict__ out, int N, int Ns,
                                                          int64_t stride)
{
    extern __shared__ double2 fsm[];   /* [256][17] */
    const int T = N >> 8;
    const int jj = threadIdx.x & 15, c = threadIdx.x >> 4;
    const int j = blockIdx.x * 16 + jj;
    const int64_t q = blockIdx.y;
    const bool live = j < T;
    const int k = j & (Ns - 1);
    double2 v[16];
    if (live) {
#pragma unroll
        for (int r1 = 0; r1 < 16; ++r1) v[r1] = fft_load<PACK>(src, q, stride, (int64_t)j + (int64_t)(c + 16 * r1) * T);
        if (Ns > 1) {
            /* input twiddles exp(SIGN 2 pi i (c + 16 r1) k / (256 Ns)) = u^c (u^16)^r1 */
            const double base = (double)k / (double)(Ns * 128);        /* 2 k / (256 Ns) */
            double sn, cs;
            sincospi(base * (double)c, &sn, &cs);
            double2 w = make_double2(cs, SIGN < 0 ? -sn : sn);
            sincospi(base * 16.0, &sn, &cs);
            const double2 u16 = make_double2(cs, SIGN < 0 ? -sn : sn);
            /* powers of u16 by sincospi of exact arguments for the power-of-two exponents, products for the others */
            double2 up[4];
            up[0] = u16;
#pragma unroll
            for (int b = 1; b < 4; ++b) {
                sincospi(base * 16.0 * (double)(1 << b), &sn, &cs);
                up[b] = make_double2(cs, SIGN < 0 ? -sn : sn);
            }
#pragma unroll
            for (int r1 = 0; r1 < 16; ++r1) {
                double2 t = w;
#pragma unroll
                for (int b = 0; b < 4; ++b)
                    if (r1 & (1 << b)) t = cmul(t, up[b]);
                v[r1] = cmul(v[r1], t);
            }
        }
        dft_small<16, SIGN>(v);    /* over r1 -> q1 */
#pragma unroll
        for (int q1 = 0; q1 < 16; ++q1) {
            double2 t = c_w256[(c * q1) & 255];
            if (SIGN > 0) t.y = -t.y;
            fsm[(c * 16 + q1) * 17 + jj] = cmul(v[q1], t);
        }
    }
    __syncthreads();
    /* second role of the thread: output residue q1 of series element j2.  While Ns < 16 consecutive outputs of ONE j are
     * adjacent in memory, so a warp takes 16 residues of two j (256-byte runs); later consecutive j are adjacent */
    const bool by_residue = Ns < 16;
    const int q1 = by_residue ? (threadIdx.x & 15) : (threadIdx.x >> 4);
    const int jj2 = by_residue ? (threadIdx.x >> 4) : (threadIdx.x & 15);
    const int j2 = blockIdx.x * 16 + jj2;
    if (j2 >= T) return;
    const int k2 = j2 & (Ns - 1);
#pragma unroll
    for (int cc = 0; cc < 16; ++cc) v[cc] = fsm[(cc * 16 + q1) * 17 + jj2];
    dft_small<16, SIGN>(v);        /* over c -> q2 */
    double2 *o = out + q * stride + (int64_t)(j2 / Ns) * Ns * 256 + k2;
#pragma unroll
    for (int q2 = 0; q2 < 16; ++q2) o[(int64_t)(q1 + 16 * q2) * Ns] = v[q2];
}

/* c_j = exp(-i pi j^2 / n) for j < n (table C) and the wrapped conj(c) of length m (table B, to be transformed) */
__global__ void __launch_bounds__(FFT_THREADS) bluestein_tables_kernel(int64_t n, int64_t m, double2 *__restrict__ C, double2 *__restrict__ B)
{
    const int64_t j = (int64_t)blockIdx.x * FFT_THREADS + threadIdx.x;
    if (j >= m) return;
    double2 b = make_double2(0.0, 0.0);
    const int64_t jj = j < n ? j : (m - j < n ? m - j : -1);     /* |index| of the wrapped chirp, or none */
    if (jj >= 0) {
        const uint64_t q = ((uint64_t)jj * (uint64_t)jj) % (uint64_t)(2 * n);
        double s, c;
        sincospi((double)q / (double)n, &s, &c);
        b = make_double2(c, s);                                   /* conj(c_jj) = exp(+i pi jj^2 / n) */
        if (j < n) C[j] = make_double2(c, -s);
    }
    B[j] = b;
}

/* A_k *= Bhat_k (grid.y = series) */
__global__ void __launch_bounds__(FFT_THREADS) fft_pointwise_kernel(double2 *__restrict__ a, const double2 *__restrict__ bhat, int64_t m)
{
    const int64_t j = (int64_t)blockIdx.x * FFT_THREADS + threadIdx.x;
    if (j >= m) return;
    double2 *p = a + (int64_t)blockIdx.y * m + j;
    *p = cmul(*p, bhat[j]);
}

/* host: the radices of a power-of-two length (16 / 4 / 2 for the bits that do not fill a byte, then 256s), and the transform itself;
 * returns the buffer (0: buf0, 1: buf1) that holds the result.  Series q starts at q * stride in both buffers.  `first`
 * (optional) replaces buf0 as the input of the first pass (fused packing). */
static inline int fft_radices(int64_t N, int *rad)
{
    int bits = 0;
    while (((int64_t)1 << bits) < N) ++bits;
    int np = 0;
    const int n256 = bits / 8;
    bits -= 8 * n256;
    /* the small radices FIRST: the first pass is the one that packs two real series into a complex one, and in a register
     * pass every thread streams through them, while the radix-256 pass would fetch them in 128-byte runs (measured: 352 us
     * against 167 us for the same pass over complex input, 256 sources x 2^17) */
    while (bits >= 4) { rad[np++] = 16; bits -= 4; }
    if (bits == 3) { rad[np++] = 4; rad[np++] = 2; }
    else if (bits == 2) rad[np++] = 4;
    else if (bits == 1) rad[np++] = 2;
    for (int i = 0; i < n256; ++i) rad[np++] = 256;
    return np;
}

#define FFT_SMEM256 (256 * 17 * sizeof(double2))

static inline int fft_setup_device()
{
    /* twiddles of the radix-256 butterfly, exp(-2 pi i e / 256), in long double; the large dynamic shared memory of its kernels */
    double2 w[256];
    for (int e = 0; e < 256; ++e) {
        const long double a = 2.0L * 3.14159265358979323846264338327950288L * (long double)e / 256.0L;
        w[e] = make_double2((double)cosl(a), (double)-sinl(a));
    }
    if (cudaMemcpyToSymbol(c_w256, w, sizeof w) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(fft_pass256_kernel<-1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT_SMEM256) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(fft_pass256_kernel<-1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT_SMEM256) != cudaSuccess) return -1;
    if (cudaFuncSetAttribute(fft_pass256_kernel<+1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)FFT_SMEM256) != cudaSuccess) return -1;
    return 0;
}

template <int SIGN>
static inline int fft_pow2(double2 *buf0, double2 *buf1, int64_t N, int64_t stride, int64_t nseries, cudaStream_t st,
                           const FftSource *first = nullptr)
{
    int rad[16];
    const int np = fft_radices(N, rad);
    int cur = 0;
    int Ns = 1;
    for (int p = 0; p < np; ++p) {
        FftSource src = {};
        const bool pack = p == 0 && first;   /* only forward transforms pack (SIGN = -1) */
        if (pack) src = *first;
        else src.in = cur ? buf1 : buf0;
        double2 *out = cur ? buf0 : buf1;
        if (rad[p] == 256) {
            const dim3 grid((unsigned)(((N >> 8) + 15) / 16), (unsigned)nseries);
            if (pack) fft_pass256_kernel<-1, true><<<grid, 256, FFT_SMEM256, st>>>(src, out, (int)N, Ns, stride);
            else fft_pass256_kernel<SIGN, false><<<grid, 256, FFT_SMEM256, st>>>(src, out, (int)N, Ns, stride);
        } else {
            const dim3 grid((unsigned)((N / rad[p] + FFT_THREADS - 1) / FFT_THREADS), (unsigned)nseries);
            if (pack) {
                if (rad[p] == 16) fft_pass_kernel<16, -1, true><<<grid, FFT_THREADS, 0, st>>>(src, out, (int)N, Ns, stride);
                else if (rad[p] == 4) fft_pass_kernel<4, -1, true><<<grid, FFT_THREADS, 0, st>>>(src, out, (int)N, Ns, stride);
                else fft_pass_kernel<2, -1, true><<<grid, FFT_THREADS, 0, st>>>(src, out, (int)N, Ns, stride);
            } else if (rad[p] == 16) fft_pass_kernel<16, SIGN, false><<<grid, FFT_THREADS, 0, st>>>(src, out, (int)N, Ns, stride);
            else if (rad[p] == 4) fft_pass_kernel<4, SIGN, false><<<grid, FFT_THREADS, 0, st>>>(src, out, (int)N, Ns, stride);
            else fft_pass_kernel<2, SIGN, false><<<grid, FFT_THREADS, 0, st>>>(src, out, (int)N, Ns, stride);
        }
        Ns *= rad[p];
        cur ^= 1;
    }
    return cur;
}
