// overlap.cu -- SURVEY.md 8(f)-1, the first "next" row: steps iv-v of the paper's likelihood evaluation:
// Fourier transform of the TDI channels, the analytic noise PSDs of Sec. II C (Eqs. 2.10-2.13) and the
// noise-weighted inner product, overlap, mismatch and SNR of Eqs. (5.1), (5.2), (6.1).
//
//   noise_psd_kernel   S_n^{A,E}(f_k), S_n^T(f_k) on f_k = k df                      (ALU, tiny)
//   fft.cuh            x~_k = sum_n x_n exp(-2 pi i k n / N), hand-written: Stockham radix-16 passes for powers of two,
//                      Bluestein's chirp-z on top of them for every other length; the A (E, T) series of the two
//                      responses ride in ONE complex transform, z = a + i b                  (HBM-bound passes)
//   products_kernel    per (source, channel, block of bins): a~_k, b~_k from Z_k and Z_{n-k}, partial sums of
//                      |a~|^2 / S, |b~|^2 / S, Re(a~* b~) / S over the band f_min <= f_k <= f_max   (HBM-bound: 32 B per bin)
//   finalize_kernel    fixed-order sum of the partials (deterministic), 4 df dt^2 scaling, overlap, mismatch, SNR
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include <algorithm>
#include <new>

#include "../../include/lisatdi.h"
#include "fft.cuh"

#define OVL_CUDA_OK(expr)                                                                                 \
    do {                                                                                                  \
        const cudaError_t e_ = (expr);                                                                    \
        if (e_ != cudaSuccess) {                                                                          \
            if (getenv("LTDI_DEBUG")) fprintf(stderr, "lisatdi %s:%d: %s\n", __FILE__, __LINE__, cudaGetErrorString(e_)); \
            (void)cudaGetLastError();                                                                     \
            return LTDI_ECUDA;                                                                            \
        }                                                                                                 \
    } while (0)
#define OVL_THREADS 256
#define OVL_BINS_PER_THREAD 8
#define OVL_BINS_PER_BLOCK (OVL_THREADS * OVL_BINS_PER_THREAD)

struct ltdi_overlap {
    int64_t n, ld, batch, chunk, nf, nblk;
    int64_t m;            /* transform length: n if it is a power of two, else the Bluestein length 2^p >= 2 n - 1 */
    bool pow2;
    size_t table_bytes, buf_bytes, part_bytes, total;   /* chirp tables | two ping-pong buffers [3 chunk][m] | partials */
};

namespace {

constexpr double kC = 299792458.0;

// Eqs. (2.10)-(2.13)
__global__ void noise_psd_kernel(ltdi_noise_desc d, double df, int64_t nf, double *__restrict__ psd)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nf) return;
    if (k == 0) { /* f = 0 lies outside every band: 1 / S = 0 */
        psd[0] = INFINITY;
        psd[nf] = INFINITY;
        return;
    }
    const double pi = 3.14159265358979323846;
    const double f = (double)k * df;
    const double x = 2.0 * pi * f * d.arm_m / kC;
    const double s_acc = 2.4e-15 * 2.4e-15, s_oms = 7.9e-12 * 7.9e-12;
    const double r1 = 0.0004 / f, r2 = f / 0.008, r3 = 0.002 / f;
    const double w1 = 2.0 * pi * f * kC, w2 = 2.0 * pi * f / kC;
    const double s_pm = s_acc / (w1 * w1) * (1.0 + r1 * r1) * (1.0 + (r2 * r2) * (r2 * r2));     /* (2.10a) */
    const double s_op = s_oms * (w2 * w2) * (1.0 + (r3 * r3) * (r3 * r3));                       /* (2.10b) */
    double gal = 0.0;
    if (d.galactic) { /* (2.11), (2.12) with T_obs in years */
        const double lt = log10(d.t_obs_yr);
        const double f1 = pow(10.0, -0.223499956 * lt - 2.70408439);
        const double fk = pow(10.0, -0.360976122 * lt - 2.37822436);
        const double sx = sin(x);
        gal = 2.0 * x * x * sx * sx * 1.28265531e-44 * pow(f, -7.0 / 3.0) * exp(-pow(f / f1, 1.62966700)) *
              (1.0 + tanh((fk - f) / 4.81078093e-4));
    }
    double sx, cx;
    sincos(x, &sx, &cx);
    const double s2x = sin(2.0 * x), c2x = cos(2.0 * x), shx = sin(0.5 * x);
    const double lam = d.gen == LTDI_GEN_20 ? 4.0 * s2x * s2x : 1.0;
    psd[k] = 8.0 * lam * sx * sx * (2.0 * (3.0 + 2.0 * cx + c2x) * s_pm + (2.0 + cx) * s_op) + 1.5 * lam * gal; /* (2.13a) */
    psd[nf + k] = 16.0 * lam * sx * sx * ((1.0 - cx) * s_op + 8.0 * (shx * shx) * (shx * shx) * s_pm) + lam * gal; /* (2.13b) */
}

// zb: [chunk][3][m] complex: the transform (Bluestein: before the final chirp C_k) of z = a_c + i b_c; part: [chunk][3][nblk][3]
__global__ void __launch_bounds__(OVL_THREADS) products_kernel(const double2 *__restrict__ zb, const double2 *__restrict__ C,
                                                               const double *__restrict__ psd, int64_t n, int64_t m, int64_t nf,
                                                               int64_t nsrc, double df, double fmin, double fmax,
                                                               int64_t nblk, double *__restrict__ part)
{
    const int c = blockIdx.y;
    const int64_t s = blockIdx.z;
    const double2 *z = zb + (s * 3 + c) * m;
    const double *sn = psd + (c == 2 ? nf : 0);
    double aa = 0.0, bb = 0.0, ab = 0.0;
    const int64_t k0 = (int64_t)blockIdx.x * OVL_BINS_PER_BLOCK + threadIdx.x;
#pragma unroll
    for (int j = 0; j < OVL_BINS_PER_THREAD; ++j) {
        const int64_t k = k0 + (int64_t)j * OVL_THREADS;
        if (k > 0 && k < nf) {
            const double f = (double)k * df;
            if (f >= fmin && f <= fmax) {                      /* (5.1): rectangle rule over the bins of the band */
                double2 zk = z[k], zn = z[n - k];
                if (C) { zk = cmul(zk, C[k]); zn = cmul(zn, C[n - k]); }
                /* a~ = (Z_k + conj Z_{n-k}) / 2, b~ = (Z_k - conj Z_{n-k}) / (2 i) */
                const double2 u = make_double2(0.5 * (zk.x + zn.x), 0.5 * (zk.y - zn.y));
                const double2 v = make_double2(0.5 * (zk.y + zn.y), -0.5 * (zk.x - zn.x));
                const double inv = 1.0 / sn[k];
                aa += (u.x * u.x + u.y * u.y) * inv;
                bb += (v.x * v.x + v.y * v.y) * inv;
                ab += (u.x * v.x + u.y * v.y) * inv;           /* Re(conj(a~) b~) */
            }
        }
    }
    (void)nsrc;
    __shared__ double red[3][OVL_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        aa += __shfl_xor_sync(0xffffffffu, aa, o);
        bb += __shfl_xor_sync(0xffffffffu, bb, o);
        ab += __shfl_xor_sync(0xffffffffu, ab, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { red[0][warp] = aa; red[1][warp] = bb; red[2][warp] = ab; }
    __syncthreads();
    if (threadIdx.x < 3) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < OVL_THREADS / 32; ++w) t += red[threadIdx.x][w];
        part[((s * 3 + c) * nblk + blockIdx.x) * 3 + threadIdx.x] = t;
    }
}

// out: [batch][3][5] = <a|a>, <b|b>, <a|b>, overlap (5.2), mismatch 1 - |O|;  snr: [batch][3] = rho_a, rho_b (6.1) and
// ln L = -1/2 <a - b|a - b> (D4).  One block of three warps per source, warp c sums the partials of channel c: lane i takes blocks i, i + 32, ...,
// then a shuffle tree -- a fixed order, so the result does not depend on the launch.
__global__ void __launch_bounds__(96) finalize_kernel(const double *__restrict__ part, int64_t nsrc, int64_t nblk,
                                                      double scale, double *__restrict__ out, double *__restrict__ snr)
{
    const int64_t s = blockIdx.x;
    const int c = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double aa = 0.0, bb = 0.0, ab = 0.0;
    const double *p = part + (s * 3 + c) * nblk * 3;
    for (int64_t i = lane; i < nblk; i += 32) { aa += p[3 * i]; bb += p[3 * i + 1]; ab += p[3 * i + 2]; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        aa += __shfl_xor_sync(0xffffffffu, aa, o);
        bb += __shfl_xor_sync(0xffffffffu, bb, o);
        ab += __shfl_xor_sync(0xffffffffu, ab, o);
    }
    aa *= scale; bb *= scale; ab *= scale;
    __shared__ double self[3][3];
    if (lane == 0) {
        const double ov = ab / (sqrt(aa) * sqrt(bb));
        double *o = out + (s * 3 + c) * 5;
        o[0] = aa; o[1] = bb; o[2] = ab; o[3] = ov; o[4] = 1.0 - fabs(ov);
        self[c][0] = aa; self[c][1] = bb; self[c][2] = ab;
    }
    __syncthreads();
    if (snr && threadIdx.x < 2) snr[3 * s + threadIdx.x] = sqrt((self[0][threadIdx.x] + self[1][threadIdx.x]) + self[2][threadIdx.x]);
    if (snr && threadIdx.x == 2) { /* (D4): ln L = -1/2 <a - b|a - b> summed over the channels */
        double q = 0.0;
        for (int ch = 0; ch < 3; ++ch) q += (self[ch][0] + self[ch][1]) - 2.0 * self[ch][2];
        snr[3 * s + 2] = -0.5 * q;
    }
    (void)nsrc;
}

size_t align256(size_t x) { return (x + 255) / 256 * 256; }

} // namespace

extern "C" {

int ltdi_noise_psd(const ltdi_noise_desc *desc, double df, int64_t nf, double *d_psd, void *stream)
{
    if (!desc || !(df > 0.0) || nf < 1 || !d_psd || !(desc->arm_m > 0.0) || !(desc->t_obs_yr > 0.0)) return LTDI_EINVAL;
    if (desc->gen != LTDI_GEN_15 && desc->gen != LTDI_GEN_20) return LTDI_EINVAL;
    noise_psd_kernel<<<(unsigned)((nf + 255) / 256), 256, 0, (cudaStream_t)stream>>>(*desc, df, nf, d_psd);
    OVL_CUDA_OK(cudaGetLastError());
    return LTDI_OK;
}

int ltdi_overlap_create(int64_t n, int64_t ld, int64_t batch, ltdi_overlap **out, size_t *work_bytes)
{
    if (n < 2 || n > ((int64_t)1 << 27) || ld < n || batch < 1 || !out || !work_bytes) return LTDI_EINVAL;
    ltdi_overlap *o = new (std::nothrow) ltdi_overlap;
    if (!o) return LTDI_EINVAL;
    o->n = n; o->ld = ld; o->batch = batch; o->nf = n / 2 + 1;
    o->pow2 = (n & (n - 1)) == 0;
    o->m = n;
    if (!o->pow2) { o->m = 1; while (o->m < 2 * n - 1) o->m <<= 1; }
    /* sources per pass: the two ping-pong buffers of a pass stay below 1 GiB (one source at least) */
    const size_t per_source = (size_t)2 * 3 * o->m * sizeof(double2);
    o->chunk = std::max<int64_t>(1, std::min<int64_t>(std::min<int64_t>(batch, 21845), (int64_t)(((size_t)1 << 30) / per_source)));
    o->nblk = (o->nf + OVL_BINS_PER_BLOCK - 1) / OVL_BINS_PER_BLOCK;
    o->table_bytes = o->pow2 ? 0 : align256((size_t)(n + 2 * o->m) * sizeof(double2));   /* C | two buffers for the chirp's transform */
    o->buf_bytes = align256((size_t)3 * o->chunk * o->m * sizeof(double2));
    o->part_bytes = align256((size_t)o->chunk * 3 * o->nblk * 3 * sizeof(double));
    o->total = o->table_bytes + 2 * o->buf_bytes + o->part_bytes;
    *work_bytes = o->total;
    *out = o;
    return LTDI_OK;
}

int ltdi_overlap_products(ltdi_overlap *o, const double *d_aA, const double *d_aE, const double *d_aT,
                          const double *d_bA, const double *d_bE, const double *d_bT, double dt, const double *d_psd,
                          double fmin, double fmax, double *d_out, double *d_snr, void *d_work, size_t work_bytes,
                          void *stream)
{
    if (!o || !d_aA || !d_aE || !d_aT || !d_bA || !d_bE || !d_bT || !d_psd || !d_out || !d_work) return LTDI_EINVAL;
    if (!(dt > 0.0) || !(fmax >= fmin)) return LTDI_EINVAL;
    if ((uintptr_t)d_work % 256) return LTDI_EINVAL;
    if (work_bytes < o->total) return LTDI_EWORKSPACE;
    {   /* per-device set-up of the transform (twiddle table, shared-memory attribute), once */
        static bool ready[64] = {};
        int dev = 0;
        OVL_CUDA_OK(cudaGetDevice(&dev));
        if (dev < 0 || dev >= 64) return LTDI_EUNSUPPORTED;
        if (!ready[dev]) {
            if (fft_setup_device()) { (void)cudaGetLastError(); return LTDI_ECUDA; }
            ready[dev] = true;
        }
    }
    cudaStream_t st = (cudaStream_t)stream;
    char *base = (char *)d_work;
    double2 *C = o->pow2 ? nullptr : (double2 *)base;
    double2 *buf0 = (double2 *)(base + o->table_bytes), *buf1 = (double2 *)(base + o->table_bytes + o->buf_bytes);
    double *part = (double *)(base + o->table_bytes + 2 * o->buf_bytes);
    const int64_t n = o->n, m = o->m;
    const double df = 1.0 / ((double)n * dt);
    /* x~ = dt * DFT(x), (5.1) rectangle rule; the Bluestein convolution carries 1 / m from its unnormalised inverse */
    const double scale = 4.0 * df * dt * dt * (o->pow2 ? 1.0 : 1.0 / ((double)m * (double)m));
    const double2 *bhat = nullptr;
    if (!o->pow2) { /* chirp tables of this length (rebuilt per call: the work area is the caller's between calls) */
        double2 *t0 = C + n, *t1 = t0 + m;
        bluestein_tables_kernel<<<(unsigned)((m + FFT_THREADS - 1) / FFT_THREADS), FFT_THREADS, 0, st>>>(n, m, C, t0);
        bhat = fft_pow2<-1>(t0, t1, m, m, 1, st) ? t1 : t0;
        OVL_CUDA_OK(cudaGetLastError());
    }
    for (int64_t b0 = 0; b0 < o->batch; b0 += o->chunk) {
        const int64_t nb = std::min(o->chunk, o->batch - b0);
        const int64_t nser = 3 * nb;
        const int64_t off = b0 * o->ld;
        /* step iv: z = a_c + i b_c (times the chirp), packed by the first pass of the transform itself */
        FftSource pack = {};
        pack.xa[0] = d_aA + off; pack.xa[1] = d_aE + off; pack.xa[2] = d_aT + off;
        pack.xb[0] = d_bA + off; pack.xb[1] = d_bE + off; pack.xb[2] = d_bT + off;
        pack.ld = o->ld; pack.n = n; pack.C = C;
        int cur = fft_pow2<-1>(buf0, buf1, m, m, nser, st, &pack);
        if (!o->pow2) {
            double2 *x = cur ? buf1 : buf0, *y = cur ? buf0 : buf1;
            fft_pointwise_kernel<<<dim3((unsigned)((m + FFT_THREADS - 1) / FFT_THREADS), (unsigned)nser), FFT_THREADS, 0, st>>>(x, bhat, m);
            cur = fft_pow2<+1>(x, y, m, m, nser, st) ? !cur : cur;
        }
        const double2 *zb = cur ? buf1 : buf0;
        const dim3 grid((unsigned)o->nblk, 3, (unsigned)nb);
        products_kernel<<<grid, OVL_THREADS, 0, st>>>(zb, C, d_psd, n, m, o->nf, nb, df, fmin, fmax, o->nblk, part);
        OVL_CUDA_OK(cudaGetLastError());
        finalize_kernel<<<(unsigned)nb, 96, 0, st>>>(part, nb, o->nblk, scale, d_out + b0 * 15,
                                                                      d_snr ? d_snr + 3 * b0 : nullptr);
        OVL_CUDA_OK(cudaGetLastError());
    }
    return LTDI_OK;
}

int ltdi_overlap_destroy(ltdi_overlap *o)
{
    if (!o) return LTDI_OK;
    delete o;
    return LTDI_OK;
}

} // extern "C"
