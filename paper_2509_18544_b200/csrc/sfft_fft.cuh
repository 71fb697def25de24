// sfft_fft.cuh -- building blocks of the FP64 Stockham FFTs of libsfft (steps a1 and a5) and of the
// asynchronous staging (bulk copies completing on mbarriers) that feeds the column and lag kernels.
//
// One power-of-two transform of length N (512 <= N <= 4096) is computed by T = N/16 threads, 16 complex
// values per thread in registers.  "Canonical" register layout: thread j holds elements j + q T,
// q = 0..15.  A Stockham (autosort) pass of radix R (R | 16) does 16/R butterflies per thread straight from
// the canonical layout -- butterfly jb = j + b T takes elements jb + m N/R, m < R -- and scatters the results
// into a shared-memory exchange buffer at position (jb div Ns) Ns R + (jb mod Ns) + m Ns, Ns = product of the
// radices of the earlier passes; after a barrier the next pass reloads the canonical layout.  The last pass
// leaves natural order in registers (v[q] = element j + q T).
//
// Exchange buffers hold 16-byte elements at XOR-swizzled positions (no padding: the column kernels need the
// 64 KB of a 4096-point column to be exactly 64 KB so that two workers and their staging rings fit one SM):
//   swz<LR0>(i) = i ^ ((i >> LR0) & (2^LR0 - 1)),  2^LR0 = radix of the FIRST pass,
// which spreads the stride-R scatter of the first pass over all banks; every later pass and every canonical
// reload touches runs of >= 8 consecutive elements, which a constant XOR only permutes.
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

// Planes (row-transformed intermediates and spectra) are stored COLUMN-MAJOR: element (ky, kx) of a plane with
// My rows at kx * My + ky, so a column is one contiguous run (bulk copies, coalesced 16-byte accesses along ky).
// Intermediates have Hx columns (column 0 = X[0] + i X[Hx], both real along x); spectra have Hx + 1 true columns
// kx = 0..Hx (the forward column pass separates the packed column once, sfft_cols.cu).
SFFT_HD size_t plane_idx(int ky, int kx, int My) { return (size_t)kx * My + ky; }

// Storage of spectra: complex128 (cplx) or, in the reduced-memory plan mode (sfft_plan_create_ex, SFFT_PLAN_FP32_SPECTRA),
// complex64 (float2); arithmetic is FP64 either way.
SFFT_HD cplx ld_c(const double2 &a) { return a; }
SFFT_HD cplx ld_c(const float2 &a) { return mk((double)a.x, (double)a.y); }
SFFT_HD void st_c(double2 *p, cplx v) { *p = v; }
SFFT_HD void st_c(float2 *p, cplx v) { float2 f; f.x = (float)v.x; f.y = (float)v.y; *p = f; }

template <int LR0> SFFT_HD int swz(int i) { return i ^ ((i >> LR0) & ((1 << LR0) - 1)); }

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

__host__ __device__ constexpr int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }

#ifdef __CUDACC__
// ---------------------------------------------------------------------------------------------
// passes (device).  X: exchange buffer of 16-byte elements; IL rows are interleaved element by element
// (IL = 2 in the row kernels, where lane parity selects one of two image rows; 1 in the column kernels),
// r = this thread's row.  tw[k] = exp(-2 pi i k / Nt), Nt >= N a power of two.
// ---------------------------------------------------------------------------------------------

// twiddle (by w^m, w = exp(DIR 2 pi i (jb mod Ns) / (Ns R))) and DFT of one radix-R butterfly
template <int R, int DIR>
__device__ __forceinline__ void bfly(cplx *x, int jb, int log2Ns, const cplx *__restrict__ tw, int Nt) {
    constexpr int LOG2R = ilog2c(R);
    if (log2Ns > 0) {
        cplx w1 = tw[(size_t)(jb & ((1 << log2Ns) - 1)) * (Nt >> (log2Ns + LOG2R))];
        if (DIR > 0) w1.y = -w1.y;
        twiddle_powers<R>(x, w1);
    }
    dftR<R, DIR>(x);
}

// the same with the butterfly's base twiddle given (persistent kernels keep it in a register: for a pass with one
// butterfly per thread it depends on the thread only)
template <int R, int DIR>
__device__ __forceinline__ void bfly_w(cplx *x, cplx w1) {
    if (DIR > 0) w1.y = -w1.y;
    twiddle_powers<R>(x, w1);
    dftR<R, DIR>(x);
}

// exchange-buffer position of output m of butterfly jb
template <int R, int LR0>
__device__ __forceinline__ int out_pos(int jb, int m, int log2Ns) {
    constexpr int LOG2R = ilog2c(R);
    const int base = ((jb >> log2Ns) << (log2Ns + LOG2R)) + (jb & ((1 << log2Ns) - 1));
    return swz<LR0>(base + (m << log2Ns));
}

// radix-R pass from the canonical registers into the exchange buffer (caller: barrier before and after)
template <int R, int DIR, int LR0, int IL>
__device__ __forceinline__ void pass_store(const cplx (&v)[16], cplx *X, int r, int j, int T, int log2Ns,
                                           const cplx *__restrict__ tw, int Nt) {
    constexpr int NBF = 16 / R;
#pragma unroll
    for (int b = 0; b < NBF; b++) {
        cplx x[R];
#pragma unroll
        for (int m = 0; m < R; m++) x[m] = v[b + m * NBF];
        const int jb = j + b * T;
        bfly<R, DIR>(x, jb, log2Ns, tw, Nt);
#pragma unroll
        for (int m = 0; m < R; m++) X[(size_t)out_pos<R, LR0>(jb, m, log2Ns) * IL + r] = x[m];
    }
}

template <int LR0, int IL>
__device__ __forceinline__ void load_canonical(cplx (&v)[16], const cplx *X, int r, int j, int T) {
#pragma unroll
    for (int q = 0; q < 16; q++) v[q] = X[(size_t)swz<LR0>(j + q * T) * IL + r];
}

// last pass (Ns R = N): results stay in the registers, natural order v[q] = element j + q T
template <int R, int DIR>
__device__ __forceinline__ void pass_regs(cplx (&v)[16], int j, int T, int log2Ns, const cplx *__restrict__ tw, int Nt) {
    constexpr int NBF = 16 / R;
#pragma unroll
    for (int b = 0; b < NBF; b++) {
        cplx x[R];
#pragma unroll
        for (int m = 0; m < R; m++) x[m] = v[b + m * NBF];
        bfly<R, DIR>(x, j + b * T, log2Ns, tw, Nt);
#pragma unroll
        for (int m = 0; m < R; m++) v[b + m * NBF] = x[m];
    }
}

// The persistent kernels derive ~50 shared-memory addresses from the thread index.  They are loop invariant, so the
// compiler hoists them out of the item loop and keeps them in registers across it -- next to 16 complex values that is
// what spilled.  An index laundered through an empty asm per item is recomputed where it is used instead.
__device__ __forceinline__ int opaque_index(int j) { asm volatile("" : "+r"(j)); return j; }

// ---------------------------------------------------------------------------------------------
// asynchronous staging: bulk global -> shared copies (TMA engine, SASS UBLKCP) completing on an mbarrier,
// and named barriers for thread groups smaller than the CTA
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *b, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// one arrival that also announces `bytes` of asynchronous copies to come (0: a plain arrival)
__device__ __forceinline__ void mbar_expect(unsigned long long *b, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
// A consumer thread hands a staging-ring slot back for refilling: the slot was read through the generic proxy and will be
// WRITTEN by the copy engine (async proxy), and nothing orders the two unless the reader says so -- a refill from L2
// takes ~150 ns, a shared-memory load queued behind another CTA's exchange phase can take longer.  The proxy fence
// makes this thread's earlier shared-memory accesses complete before anything the async proxy does after the arrival.
// (Without it: a handful of wrong spectrum elements per 4088 x 4088 frame, run-to-run different; bar.sync does not
// order the copy engine either.  tests/test_gpu_fullsize.py::test_run_to_run_reproducibility_at_full_size.)
__device__ __forceinline__ void slot_release(unsigned long long *b) {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_inval(unsigned long long *b) {
    asm volatile("mbarrier.inval.shared::cta.b64 [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *b, unsigned parity) {
    asm volatile("{\n.reg .pred p;\nWAIT_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}\n"
                 ::"r"(smem_u32(b)), "r"(parity) : "memory");
}
// bytes: a multiple of 16; both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gsrc, unsigned bytes, unsigned long long *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void bulk_s2g(void *gdst, const void *smem_src, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory"); }
template <int N> __device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group %0;" ::"n"(N) : "memory"); }
// writes of this thread to shared memory become visible to the asynchronous (bulk copy) proxy
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// barrier `id` (1..15) over `count` threads (a multiple of 32); id 0 is __syncthreads()
__device__ __forceinline__ void group_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
#endif

} // namespace sfft
