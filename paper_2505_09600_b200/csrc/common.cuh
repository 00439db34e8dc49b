// common.cuh -- shared declarations of the CUDA path (sm_100a, fp64).
//
// Notation follows arXiv 2505.09600: links l = +1,+2,+3,-1,-2,-3 (index 0..5), spacecraft
// 1,2,3 (index 0..2), y_slr single-link responses, X,Y,Z Michelson, A,E,T (Eq. 2.9).
// "P:n" = PAPER.md line n, "G<k>" = reading k in DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

#include "../../include/lisatdi.h"
#include "../../include/lisatdi_bench.h"

#define LTDI_C_LIGHT 299792458.0 /* m/s */
#define LTDI_MAX_TAPS 64
#define LTDI_FRAME_STRIDE 16 /* doubles per source in the frame buffer */

struct ltdi_orbits {
    ltdi_orbit_desc desc;
    const double *d_tab; /* [LTDI_TABLE_ROWS][stride] */
    int64_t stride;
    const double *d_anc; /* TDI weight anchors and their headers from ltdi_orbits_prepare(), or NULL */
    int anc_gen, anc_M;  /* generation and tap count they were computed for */
    bool anc_has2;       /* they carry the second derivative of the weights too */
};

/* table rows: LTDI_TABLE_ROWS rows of doubles, then LTDI_TABLE_LO_ROWS rows of floats (same row stride in elements)
 * with the low parts of the double-double n_l and L_l (orbit.cuh) */
enum { ROW_R = 0, ROW_N = 9, ROW_L = 18 };
enum { LO_N = 0, LO_L = 9 };
#define LTDI_TABLE_LO_ROWS 16
#define LTDI_TABLE_BYTES_PER_SAMPLE (LTDI_TABLE_ROWS * 8 + LTDI_TABLE_LO_ROWS * 4)

/* sender / receiver spacecraft (0-based) of link index 0..5 */
__host__ __device__ __forceinline__ int link_sender(int l)
{
    /* +1: 3->2, +2: 1->3, +3: 2->1, -1: 2->3, -2: 3->1, -3: 1->2 */
    return l < 3 ? (l + 2) % 3 : (l - 3 + 1) % 3;
}
__host__ __device__ __forceinline__ int link_receiver(int l)
{
    return l < 3 ? (l + 1) % 3 : (l - 3 + 2) % 3;
}

struct Margins {
    int64_t m1; /* reach of the projection (both sides) */
    int64_t m2; /* backward reach of the TDI stage */
    int64_t w;  /* stencil half width */
    int64_t lo, hi;
};

/* The library is one translation unit (lisatdi.cu includes the .cuh files), so that the
 * __constant__ tables below are visible to every kernel without relocatable device code. */

/* Lagrange denominators 1 / prod_{m != k} (k - m) for every even tap count M = 2 (r + 1):
 * row r, column k + M/2 - 1 */
__constant__ double c_lag_inv_den[32 * LTDI_MAX_TAPS];

/* a failed CUDA call becomes LTDI_ECUDA; with LTDI_DEBUG set in the environment the CUDA error is printed */
#define LTDI_CUDA_OK(expr)                                                                              \
    do {                                                                                                \
        const cudaError_t ltdi_err_ = (expr);                                                           \
        if (ltdi_err_ != cudaSuccess) {                                                                 \
            if (getenv("LTDI_DEBUG"))                                                                   \
                fprintf(stderr, "lisatdi %s:%d: %s\n", __FILE__, __LINE__, cudaGetErrorString(ltdi_err_)); \
            (void)cudaGetLastError();                                                                   \
            return LTDI_ECUDA;                                                                          \
        }                                                                                               \
    } while (0)
