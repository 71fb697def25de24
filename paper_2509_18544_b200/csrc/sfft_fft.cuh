// sfft_fft.cuh -- register/shared-memory Stockham FFT building blocks (FP64 complex).
//
// One power-of-two FFT of length N (32 <= N <= 8192) is computed by T = N/16 threads.
// Every thread holds 16 complex values v[0..15] in registers.  "Canonical" register
// layout: thread j holds elements j + q*T, q = 0..15.  A pass of radix R (16, or the
// remaining factor 2/4/8 in the last pass) does 16/R butterflies per thread straight from
// the canonical layout, scatters the results into shared memory at the Stockham
// (autosort) positions, and after a barrier the next pass reloads the canonical layout.
// The last pass leaves its results canonical in registers (natural order: v[q] is
// element j + q*T), so the caller stores them wherever it wants (global memory for
// column passes, shared memory for the real<->complex untangle of row passes).
//
// Shared-memory indices are padded by one element per 16 (phys = i + i/16) so that the
// stride-16 scatter of the first pass is bank-conflict free for 16-byte accesses.
//
// The functions are __host__ __device__ so that the index arithmetic can be exercised on
// the CPU by tests (tests/test_fft_host.py builds a host emulation of the passes).
#pragma once
#include <cuda_runtime.h>

#ifndef SFFT_HD
#define SFFT_HD __host__ __device__ __forceinline__
#endif

namespace sfft {

typedef double2 cplx;

SFFT_HD cplx mk(double x, double y) { cplx r; r.x = x; r.y = y; return r; }
SFFT_HD cplx cadd(cplx a, cplx b) { return mk(a.x + b.x, a.y + b.y); }
SFFT_HD cplx csub(cplx a, cplx b) { return mk(a.x - b.x, a.y - b.y); }
SFFT_HD cplx cmul(cplx a, cplx b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
SFFT_HD cplx cmulc(cplx a, cplx b) { /* conj(a) * b */ return mk(a.x * b.x + a.y * b.y, a.x * b.y - a.y * b.x); }
SFFT_HD cplx cconj(cplx a) { return mk(a.x, -a.y); }
SFFT_HD cplx cscale(cplx a, double s) { return mk(a.x * s, a.y * s); }
// multiply by DIR*i  (W4 = exp(DIR*2*pi*i/4))
template <int DIR> SFFT_HD cplx mul_w4(cplx a) { return DIR > 0 ? mk(-a.y, a.x) : mk(a.y, -a.x); }

// Spectra are stored TILE-MAJOR: column tiles of 2 adjacent kx, rows contiguous inside a tile,
//   element (ky, kx) of a My x Hx spectrum  ->  ((kx >> 1) * My + ky) * 2 + (kx & 1).
// The column pass then writes (and the subtraction reads) whole 128-byte lines -- scattered 32-byte
// sector stores of the row-major layout ran at a quarter of the line-store rate -- and the lag pass
// still finds the two columns of a tile in one 32-byte sector.
SFFT_HD size_t spec_idx(int ky, int kx, int My) { return ((size_t)(kx >> 1) * My + ky) * 2 + (kx & 1); }

SFFT_HD int pad16(int i) { return i + (i >> 4); }
SFFT_HD int padded_len(int N) { return N + (N >> 4); }

template <int DIR> SFFT_HD void dft2(cplx &a0, cplx &a1) {
    cplx t = a0; a0 = cadd(t, a1); a1 = csub(t, a1);
}

template <int DIR> SFFT_HD void dft4(cplx &a0, cplx &a1, cplx &a2, cplx &a3) {
    cplx t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = mul_w4<DIR>(csub(a1, a3));
    a0 = cadd(t0, t2); a1 = cadd(t1, t3); a2 = csub(t0, t2); a3 = csub(t1, t3);
}

#define SFFT_C1 0.92387953251128673848 /* cos(pi/8) */
#define SFFT_S1 0.38268343236508978178 /* sin(pi/8) */
#define SFFT_R2 0.70710678118654752440 /* sqrt(1/2) */

// x[0..7] natural order in, natural order out.  n = n1 + 2 n2, k = 4 k1 + k2.
template <int DIR> SFFT_HD void dft8(cplx *x) {
    dft4<DIR>(x[0], x[2], x[4], x[6]); // A[0][k2] at x[2 k2]
    dft4<DIR>(x[1], x[3], x[5], x[7]); // A[1][k2] at x[1 + 2 k2]
    x[3] = cmul(x[3], mk(SFFT_R2, DIR * SFFT_R2));
    x[5] = mul_w4<DIR>(x[5]);
    x[7] = cmul(x[7], mk(-SFFT_R2, DIR * SFFT_R2));
    cplx t[8];
#pragma unroll
    for (int k2 = 0; k2 < 4; k2++) {
        t[k2] = cadd(x[2 * k2], x[2 * k2 + 1]);
        t[k2 + 4] = csub(x[2 * k2], x[2 * k2 + 1]);
    }
#pragma unroll
    for (int k = 0; k < 8; k++) x[k] = t[k];
}

// x[0..15] natural order in, natural order out.  n = n1 + 4 n2, k = 4 k1 + k2.
template <int DIR> SFFT_HD void dft16(cplx *x) {
#pragma unroll
    for (int n1 = 0; n1 < 4; n1++) dft4<DIR>(x[n1], x[n1 + 4], x[n1 + 8], x[n1 + 12]); // A[n1][k2] at x[n1+4k2]
    // twiddles W16^(n1*k2)
    x[1 + 4 * 1] = cmul(x[1 + 4 * 1], mk(SFFT_C1, DIR * SFFT_S1));   // W^1
    x[1 + 4 * 2] = cmul(x[1 + 4 * 2], mk(SFFT_R2, DIR * SFFT_R2));   // W^2
    x[1 + 4 * 3] = cmul(x[1 + 4 * 3], mk(SFFT_S1, DIR * SFFT_C1));   // W^3
    x[2 + 4 * 1] = cmul(x[2 + 4 * 1], mk(SFFT_R2, DIR * SFFT_R2));   // W^2
    x[2 + 4 * 2] = mul_w4<DIR>(x[2 + 4 * 2]);                        // W^4
    x[2 + 4 * 3] = cmul(x[2 + 4 * 3], mk(-SFFT_R2, DIR * SFFT_R2));  // W^6
    x[3 + 4 * 1] = cmul(x[3 + 4 * 1], mk(SFFT_S1, DIR * SFFT_C1));   // W^3
    x[3 + 4 * 2] = cmul(x[3 + 4 * 2], mk(-SFFT_R2, DIR * SFFT_R2));  // W^6
    x[3 + 4 * 3] = cmul(x[3 + 4 * 3], mk(-SFFT_C1, -DIR * SFFT_S1)); // W^9
#pragma unroll
    for (int k2 = 0; k2 < 4; k2++) dft4<DIR>(x[4 * k2], x[4 * k2 + 1], x[4 * k2 + 2], x[4 * k2 + 3]); // X[4k1+k2] at x[k1+4k2]
    cplx t[16];
#pragma unroll
    for (int k = 0; k < 16; k++) t[k] = x[k];
#pragma unroll
    for (int k1 = 0; k1 < 4; k1++)
#pragma unroll
        for (int k2 = 0; k2 < 4; k2++) x[4 * k1 + k2] = t[k1 + 4 * k2];
}

template <int R, int DIR> SFFT_HD void dftR(cplx *x) {
    if (R == 16) dft16<DIR>(x);
    else if (R == 8) dft8<DIR>(x);
    else if (R == 4) dft4<DIR>(x[0], x[1], x[2], x[3]);
    else dft2<DIR>(x[0], x[1]);
}

// x[m] *= w^m, m = 1..R-1, powers built by a depth-4 product tree (<= 4 roundings deep).
template <int R> SFFT_HD void twiddle_powers(cplx *x, cplx w1) {
    cplx w2 = cmul(w1, w1);
    x[1] = cmul(x[1], w1);
    if (R >= 4) {
        cplx w3 = cmul(w2, w1);
        x[2] = cmul(x[2], w2);
        x[3] = cmul(x[3], w3);
        if (R >= 8) {
            cplx w4 = cmul(w2, w2), w5 = cmul(w4, w1), w6 = cmul(w3, w3), w7 = cmul(w4, w3);
            x[4] = cmul(x[4], w4); x[5] = cmul(x[5], w5); x[6] = cmul(x[6], w6); x[7] = cmul(x[7], w7);
            if (R >= 16) {
                cplx w8 = cmul(w4, w4);
                x[8] = cmul(x[8], w8);
                x[9] = cmul(x[9], cmul(w8, w1));
                x[10] = cmul(x[10], cmul(w5, w5));
                x[11] = cmul(x[11], cmul(w8, w3));
                x[12] = cmul(x[12], cmul(w6, w6));
                x[13] = cmul(x[13], cmul(w8, w5));
                x[14] = cmul(x[14], cmul(w7, w7));
                x[15] = cmul(x[15], cmul(w8, w7));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Generic form: E values per thread (E = 8 or 16), T = N/E threads per transform.  Canonical layout:
// thread j holds elements j + q*T, q = 0..E-1.  Shared-memory indices are padded by one element per E
// (phys = i + i/E) so that the stride-E scatter of the first pass is bank-conflict free.
// ---------------------------------------------------------------------------------------------
template <int E> SFFT_HD int padE(int i) { return i + i / E; }
template <int E> SFFT_HD int padded_lenE(int N) { return N + N / E; }

// One Stockham pass of radix R (R divides E) on the canonical registers of thread j.
//   Ns = product of the radices of earlier passes (log2Ns given), tw[k] = exp(-2 pi i k/Nt).
// STORE: results go to shared memory s (padded) at their autosort positions; otherwise (last pass)
// they stay canonical in v.
template <int E, int R, int DIR, bool STORE>
SFFT_HD void fft_passE(cplx *v, cplx *s, int j, int T, int log2Ns, const cplx *tw, int Nt) {
    constexpr int NBF = E / R; // butterflies per thread
    constexpr int LOG2R = (R == 16) ? 4 : (R == 8) ? 3 : (R == 4) ? 2 : 1;
    const int Ns = 1 << log2Ns;
#pragma unroll
    for (int b = 0; b < NBF; b++) {
        cplx x[R];
#pragma unroll
        for (int m = 0; m < R; m++) x[m] = v[b + m * NBF];
        const int jb = j + b * T;
        const int k = jb & (Ns - 1);
        if (log2Ns > 0) {
            cplx w1 = tw[(size_t)k * (Nt >> (log2Ns + LOG2R))];
            if (DIR > 0) w1.y = -w1.y;
            twiddle_powers<R>(x, w1);
        }
        dftR<R, DIR>(x);
        if (STORE) {
            const int base = ((jb >> log2Ns) << (log2Ns + LOG2R)) + k;
#pragma unroll
            for (int m = 0; m < R; m++) s[padE<E>(base + (m << log2Ns))] = x[m];
        } else {
#pragma unroll
            for (int m = 0; m < R; m++) v[b + m * NBF] = x[m];
        }
    }
}

template <int E> SFFT_HD void fft_load_canonicalE(cplx *v, const cplx *s, int j, int T) {
#pragma unroll
    for (int q = 0; q < E; q++) v[q] = s[padE<E>(j + q * T)];
}

#ifdef __CUDACC__
// Whole FFT of length N = 2^log2N >= 2E for the T = N/E threads of one transform inside a CTA in which
// EVERY thread calls this with the same N (barriers are CTA-wide).  v canonical in, canonical out.
// LOG2N_CT != 0 fixes the length at compile time (the hot sizes): every shift, mask, padded index and
// twiddle stride below then folds to a constant and the passes unroll, which removes most of the
// integer instructions that otherwise outnumber the FP64 ones.
template <int DIR, int E, int LOG2N_CT = 0>
__device__ __forceinline__ void fft_blockE(cplx *v, cplx *s, int log2N_rt, int j, const cplx *tw, int Nt) {
    constexpr int LOG2E = (E == 16) ? 4 : 3;
    const int log2N = LOG2N_CT ? LOG2N_CT : log2N_rt;
    const int T = 1 << (log2N - LOG2E);
    __syncthreads();
    fft_passE<E, E, DIR, true>(v, s, j, T, 0, tw, Nt);
    __syncthreads();
    fft_load_canonicalE<E>(v, s, j, T);
    if (LOG2N_CT) {
        // up to two more full-radix passes (N <= E^4), all bounds known
        if (LOG2E + LOG2E < log2N) {
            __syncthreads();
            fft_passE<E, E, DIR, true>(v, s, j, T, LOG2E, tw, Nt);
            __syncthreads();
            fft_load_canonicalE<E>(v, s, j, T);
        }
        if (3 * LOG2E < log2N) {
            __syncthreads();
            fft_passE<E, E, DIR, true>(v, s, j, T, 2 * LOG2E, tw, Nt);
            __syncthreads();
            fft_load_canonicalE<E>(v, s, j, T);
        }
        const int log2Ns = (3 * LOG2E < log2N) ? 3 * LOG2E : (2 * LOG2E < log2N) ? 2 * LOG2E : LOG2E;
        switch (log2N - log2Ns) {
        case 4: if (E >= 16) fft_passE<E, (E >= 16 ? 16 : E), DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
        case 3: fft_passE<E, 8, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
        case 2: fft_passE<E, 4, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
        default: fft_passE<E, 2, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
        }
        return;
    }
    int log2Ns = LOG2E;
#pragma unroll 1
    while (log2Ns + LOG2E < log2N) {
        __syncthreads();
        fft_passE<E, E, DIR, true>(v, s, j, T, log2Ns, tw, Nt);
        __syncthreads();
        fft_load_canonicalE<E>(v, s, j, T);
        log2Ns += LOG2E;
    }
    switch (log2N - log2Ns) {
    case 4: if (E >= 16) fft_passE<E, (E >= 16 ? 16 : E), DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
    case 3: fft_passE<E, 8, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
    case 2: fft_passE<E, 4, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
    default: fft_passE<E, 2, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
    }
}
#endif

// One Stockham pass of radix R on the canonical registers of thread j.
//   N = FFT length, T = N/16, Ns = product of the radices of earlier passes (log2Ns given),
//   tw[k] = exp(-2 pi i k / Nt) (Nt >= N, power of two).
// If STORE, results go to shared memory s (padded) at their autosort positions (the caller
// puts a barrier before -- all threads must have finished reading s -- and after);
// otherwise (last pass, Ns*R == N) they stay canonical in v.
template <int R, int DIR, bool STORE>
SFFT_HD void fft_pass(cplx *v, cplx *s, int j, int T, int log2Ns, const cplx *tw, int Nt) {
    constexpr int NB = 16 / R; // butterflies per thread
    constexpr int LOG2R = (R == 16) ? 4 : (R == 8) ? 3 : (R == 4) ? 2 : 1;
    const int Ns = 1 << log2Ns;
#pragma unroll
    for (int b = 0; b < NB; b++) {
        cplx x[R];
#pragma unroll
        for (int m = 0; m < R; m++) x[m] = v[b + m * NB];
        const int jb = j + b * T;
        const int k = jb & (Ns - 1);
        if (log2Ns > 0) {
            // exp(DIR * 2 pi i k / (Ns R)) from the table of exp(-2 pi i ./Nt)
            cplx w1 = tw[(size_t)k * (Nt >> (log2Ns + LOG2R))];
            if (DIR > 0) w1.y = -w1.y;
            twiddle_powers<R>(x, w1);
        }
        dftR<R, DIR>(x);
        if (STORE) {
            const int base = ((jb >> log2Ns) << (log2Ns + LOG2R)) + k;
#pragma unroll
            for (int m = 0; m < R; m++) s[pad16(base + (m << log2Ns))] = x[m];
        } else {
#pragma unroll
            for (int m = 0; m < R; m++) v[b + m * NB] = x[m];
        }
    }
}

SFFT_HD void fft_load_canonical(cplx *v, const cplx *s, int j, int T) {
#pragma unroll
    for (int q = 0; q < 16; q++) v[q] = s[pad16(j + q * T)];
}

#ifdef __CUDACC__
// Whole FFT for the T = N/16 threads of one transform inside a CTA in which EVERY thread
// calls this function with the same N (all barriers are CTA-wide).  v: canonical input,
// on return canonical output (natural order).  s: this transform's shared-memory region of
// padded_len(N) elements.
template <int DIR>
__device__ __forceinline__ void fft_block(cplx *v, cplx *s, int log2N, int j, const cplx *tw, int Nt) {
    const int T = 1 << (log2N - 4);
    int log2Ns = 0;
    // first pass: radix 16, no twiddles
    __syncthreads();
    fft_pass<16, DIR, true>(v, s, j, T, 0, tw, Nt);
    __syncthreads();
    fft_load_canonical(v, s, j, T);
    log2Ns = 4;
#pragma unroll 1
    while (log2Ns + 4 < log2N) {
        __syncthreads();
        fft_pass<16, DIR, true>(v, s, j, T, log2Ns, tw, Nt);
        __syncthreads();
        fft_load_canonical(v, s, j, T);
        log2Ns += 4;
    }
    switch (log2N - log2Ns) {
    case 4: fft_pass<16, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
    case 3: fft_pass<8, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
    case 2: fft_pass<4, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
    default: fft_pass<2, DIR, false>(v, s, j, T, log2Ns, tw, Nt); break;
    }
}
#endif

} // namespace sfft
