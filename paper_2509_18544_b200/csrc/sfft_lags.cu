// sfft_lags.cu -- step a2 (BASELINE.json north_star (b)):
// cross-correlations X(a,b)[du,dv] = sum_{x,y} a(x,y) b((x+du) mod nx, (y+dv) mod ny) of the
// polynomial-weighted images, read off at the kernel-offset pairs only, from the spectra.
//
//   X_M(a,b)[du,dv] = 1/(Mx My) sum_{ky} sum_{kx=0..Hx} g(kx) Re( conj(A) B e^{2 pi i (kx du/Mx + ky dv/My)} )
//
// (g = 1 for kx = 0, Hx, else 2: Hermitian symmetry of real images) is the Mx x My-circular
// correlation of the ZERO-PADDED images.  It is turned into the nx x ny-circular correlation
// the method defines (reading C6) by adding the few products that wrap differently:
//   X_N - X_M = sum over pixels with x+du or y+dv outside the frame of
//               a(x,y) * ( b((x+du) mod nx, (y+dv) mod ny) - bpad((x+du) mod Mx, (y+dv) mod My) ).
// The product spectrum and the correlation image are never materialised: the inverse
// transform is pruned to the (2W+1)^2 lags that are used (output-pruned DFT).
//
// Kernels:
//   lagcol_kernel  stage 1: Q[p][dv][kx] = sum_ky conj(A)B e^{2 pi i ky dv/My}, kx = 0..Hx; stages of the spectra arrive
//                  by TMA (cp.async.bulk.tensor, one elected thread) in a shared-memory ring shared by all pairs
//   (sfft_border.cu) the wrap corrections X_N - X_M from border strips
//   lagrow_kernel  stage 2: lag[p][dv][du] = 1/(Mx My) sum_kx g Re(Q e^{2 pi i kx du/Mx}) + border
#include <cuda.h>
#include <new>
#include "sfft_internal.h"

namespace sfft {

constexpr int LC_NA = 16;  // decimation factor: ky = b + (My/16) a, a = 0..15
constexpr int LC_NB = 8;   // consecutive b per stage and per (pair, kx): one 128-byte line of a spectrum column
constexpr int LC_PRE = 2;  // prefetch distance in stages; the wide form uses 1 (measured there: 1 -> 0.365, 2 -> 0.374, 3 -> 0.486 ms;
                           // the two-CTA forms: 2 is 1-1.5 % faster than 1): more loads in flight are slower

struct LagMaps { CUtensorMap t; CUtensorMap s[NSCI]; };

__device__ __forceinline__ void tma_load4(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, int c3, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_load3(void *dst, const CUtensorMap *tm, int c0, int c1, int c2, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst)), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

// Stage 1, output-pruned inverse DFT along ky by decimation:
//   Q[dv] = sum_ky P[ky] e^{2 pi i ky dv/My},  P = conj(A) B,  ky = b + Tb a  (Tb = My/16)
//         = sum_b e^{2 pi i b dv/My} F_b[dv mod 16],   F_b[m] = sum_a P[b + Tb a] e^{2 pi i a m/16}.
// A thread owns (pair, kx, b mod 8): per b it forms the 16 products, runs one register-resident 16-point DFT
// and folds the outputs it needs (DLO <= dv <= DHI) into its accumulators with one complex multiply-add each:
// ~19 FP64 instructions per spectrum element and pair instead of 4 + 4 (2W+1) of the direct sum.  The eight
// b-lanes of a (pair, kx) are summed by shuffles at the end.
// Spectra are column-major, so the 8 consecutive b of one (spectrum, kx, a) are one 128-byte line: a stage is the
// TMA box {8 b, 16 a, KXC kx, all template spectra} (+ one box per science spectrum) + the 8 W phase factors,
// landing as [spectrum][kx][a][b]; stages form a ring with full/done mbarriers, thread 0 issues.
// grid = (pair groups * lag halves, kx blocks, b splits); block = npg * KXC * 8 threads.
template <int DLO, int DHI>
__device__ __forceinline__ void lag_fold(const cplx *x, const cplx *ph, cplx *acc) {
#pragma unroll
    for (int d = DLO; d <= DHI; d++) {
        const cplx v = x[((d % 16) + 16) % 16];
        cplx &a = acc[d - DLO];
        if (d == 0) { a.x += v.x; a.y += v.y; }
        else {
            const cplx e = ph[((d > 0 ? d : -d) - 1) * LC_NB];   // exp(-i phi |d|): cos = e.x, sin = -e.y
            const double c = e.x, sn = d > 0 ? -e.y : e.y;  // multiply by exp(+i phi d)
            a.x = fma(v.x, c, a.x); a.x = fma(-v.y, sn, a.x);
            a.y = fma(v.x, sn, a.y); a.y = fma(v.y, c, a.y);
        }
    }
}

struct LagArgs {
    int ns, nsci;        // spectra per stage (NK + nsci); science spectra among them (0 for Omega)
    int npg, KXC, W, nbs, nst; // pairs per group, kx per CTA, lag bound, b per split, ring stages
    int nkb;             // kx chunks of the pass (a CTA takes chunks blockIdx.y, blockIdx.y + gridDim.y, ...)
    int phW;             // lag bound of the phase table PH[b/8][d-1][b%8], d = 1..phW
};

template <int DLO, int DHI, typename ST, bool SELF = false, int PRE = LC_PRE>
__device__ __forceinline__ void lagcol_body(const LagMaps &maps, const LagArgs &la, const PairList &pl, int group, int kb, int zsplit,
                                            const cplx *__restrict__ PH, cplx *__restrict__ Q, const Geom &g,
                                            unsigned char *tile, unsigned long long *full, unsigned long long *done) {
    const int Hx = g.Hx, Tb = g.My / LC_NA, KXC = la.KXC, W = la.W, NK = g.NK;
    const int col_elems = LC_NA * LC_NB;                       // one (spectrum, kx) of a stage: 128 elements of ST
    // a stage: the spectra part in ST elements, then the phase factors (cplx); sized in bytes
    const unsigned spec_bytes = (unsigned)(la.ns * KXC * col_elems * sizeof(ST)), stage_bytes = spec_bytes + (unsigned)(la.phW * LC_NB * sizeof(cplx));
    const int kx0 = kb * KXC;           // (the pair group is the FASTEST grid index: the groups of one kx chunk run side by
                                        //  side and the second reads the chunk's spectra from L2, not from DRAM again)
    const int b0 = zsplit * la.nbs, b1 = min(Tb, b0 + la.nbs);
    const int nIt = max(0, (b1 - b0) / LC_NB);
    const int bl = threadIdx.x & (LC_NB - 1), u = threadIdx.x >> 3;
    const int lp = u / KXC, kxl = u - lp * KXC;
    const int slot = group * la.npg + lp;
    const bool active = (slot < pl.np) && (lp < la.npg);
    const int p = active ? pl.ord[slot] : 0;
    const int sa = active ? pl.a[p] : 0, sb = active ? pl.b[p] : 0;
    constexpr int NACC = DHI - DLO + 1;
    cplx acc[NACC];
#pragma unroll
    for (int d = 0; d < NACC; d++) acc[d] = mk(0.0, 0.0);

    if (threadIdx.x == 0) {
        for (int k = 0; k < la.nst; k++) { mbar_init(&full[k], 1); mbar_init(&done[k], blockDim.x); }
        mbar_fence_init();
    }
    __syncthreads();
    auto issue = [&](int it) { // thread 0
        unsigned char *st = tile + (size_t)(it % la.nst) * stage_bytes;
        unsigned long long *bar = &full[it % la.nst];
        const int b = b0 + it * LC_NB;
        mbar_expect(bar, stage_bytes);
        tma_load4(st, &maps.t, 2 * b, 0, kx0, 0, bar);
        for (int i = 0; i < la.nsci; i++) tma_load3(reinterpret_cast<ST *>(st) + (size_t)(NK + i) * KXC * col_elems, &maps.s[i], 2 * b, 0, kx0, bar);
        if (la.phW > 0) bulk_g2s(st + spec_bytes, PH + (size_t)(b / LC_NB) * la.phW * LC_NB, (unsigned)(la.phW * LC_NB * 16), bar);
    };
    if (threadIdx.x == 0)
        for (int it = 0; it < PRE && it < nIt; it++) issue(it);
    for (int it = 0; it < nIt; it++) {
        const int st_i = it % la.nst;
        if (threadIdx.x == 0 && it + PRE < nIt) {
            const int nx_i = it + PRE;
            if (nx_i >= la.nst) mbar_wait(&done[nx_i % la.nst], (unsigned)((nx_i / la.nst) - 1) & 1u); // its previous use has been consumed
            issue(nx_i);
        }
        mbar_wait(&full[st_i], (unsigned)(it / la.nst) & 1u);
        if (active) {
            const unsigned char *st = tile + (size_t)st_i * stage_bytes;
            const ST *pa = reinterpret_cast<const ST *>(st) + (size_t)(sa * KXC + kxl) * col_elems + bl;
            const ST *pb = reinterpret_cast<const ST *>(st) + (size_t)(sb * KXC + kxl) * col_elems + bl;
            cplx x[LC_NA];
            if (SELF && sa == sb) {   // a self-pair (whole warps of them: PairList::ord): |A|^2, one operand read
#pragma unroll
                for (int a = 0; a < LC_NA; a++) { const cplx z = ld_c(pa[a * LC_NB]); x[a] = mk(fma(z.x, z.x, z.y * z.y), 0.0); }
            } else {
#pragma unroll
                for (int a = 0; a < LC_NA; a++) x[a] = cmulc(ld_c(pa[a * LC_NB]), ld_c(pb[a * LC_NB]));
            }
            dft16<1>(x);
            lag_fold<DLO, DHI>(x, reinterpret_cast<const cplx *>(st + spec_bytes) + bl, acc);
        }
        slot_release(&done[st_i]);
    }
    // sum over the 8 b-lanes, then lane 0 of each (pair, kx) writes its lags
#pragma unroll
    for (int d = 0; d < NACC; d++) {
#pragma unroll
        for (int off = 1; off < LC_NB; off <<= 1) {
            acc[d].x += __shfl_xor_sync(0xffffffffu, acc[d].x, off);
            acc[d].y += __shfl_xor_sync(0xffffffffu, acc[d].y, off);
        }
    }
    const int kx = kx0 + kxl;
    if (active && bl == 0 && kx <= Hx) {
        cplx *q = Q + ((size_t)(zsplit * pl.np + p) * (2 * W + 1)) * (Hx + 1) + kx;
#pragma unroll
        for (int d = DLO; d <= DHI; d++)
            if (d >= -W && d <= W) q[(size_t)(W + d) * (Hx + 1)] = acc[d - DLO];
    }
}

// WB <= 10: one thread folds all 2 WB + 1 lags.  WB = 20: the lag range is split in two halves
// (blockIdx.x parity) to keep the accumulators in registers; both halves write disjoint rows of Q.
template <int WB, typename ST>
__global__ void __launch_bounds__(192, 2)
lagcol_kernel(const __grid_constant__ LagMaps maps, LagArgs la, PairList pl, const cplx *__restrict__ PH, cplx *__restrict__ Q, Geom g) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ unsigned long long full[4], done[4];
    unsigned char *tile = smem_raw;
    // A CTA normally takes one kx chunk (gridDim.y = nkb).  While a factorisation runs beside the pass the grid is capped
    // (run_lagcol) and the CTAs loop: a grid of 1025 short-lived CTAs would hold every SM for one CTA lifetime (57 us at
    // 4088^2) before the first slot frees, and the factorisation's next small launch waits exactly that long.
    for (int kb = blockIdx.y; kb < la.nkb; kb += gridDim.y) {
        if (WB > 10) {
            const int half = blockIdx.x & 1, grp = blockIdx.x >> 1;   // (the lag halves too: fastest index, shared L2 reads)
            if (half == 0) lagcol_body<0, WB, ST>(maps, la, pl, grp, kb, blockIdx.z, PH, Q, g, tile, full, done);
            else lagcol_body<-WB, -1, ST>(maps, la, pl, grp, kb, blockIdx.z, PH, Q, g, tile, full, done);
        } else {
            lagcol_body<-WB, WB, ST>(maps, la, pl, blockIdx.x, kb, blockIdx.z, PH, Q, g, tile, full, done);
        }
        if (kb + (int)gridDim.y < la.nkb) {   // the barriers start over with the next chunk
            __syncthreads();
            if (threadIdx.x == 0)
                for (int k = 0; k < la.nst; k++) { mbar_inval(&full[k]); mbar_inval(&done[k]); }
        }
    }
}

// The WIDE form: when the pairs of a pass need more than 192 threads but fit 384 (the Omega pass of DK = 2: 21 pairs x 2 kx
// x 8 b-lanes = 352 threads at 168 registers), ONE CTA per SM takes them all and one ring feeds them, instead of two CTAs
// that each bring their own copy of every stage from L2: 0.420 -> 0.372 ms at 4088^2 (a fifth of the warps' stall samples
// had been waiting for stage data).
template <int WB, typename ST>
__global__ void __launch_bounds__(384, 1)
lagcol_wide_kernel(const __grid_constant__ LagMaps maps, LagArgs la, PairList pl, const cplx *__restrict__ PH, cplx *__restrict__ Q, Geom g) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ unsigned long long full[4], done[4];
    lagcol_body<-WB, WB, ST, true, 1>(maps, la, pl, blockIdx.x, blockIdx.y, blockIdx.z, PH, Q, g, smem_raw, full, done);
}

// phase table PH[b/8][d-1][b%8] = exp(-2 pi i b d/My), b < My/16, d = 1..W (W = the kernel's compile-time lag bound WB)
__global__ void lag_phase_kernel(cplx *PH, int W, int My, const cplx *__restrict__ tw, int Nt) {
    const int id = blockIdx.x * blockDim.x + threadIdx.x, Tb = My / LC_NA;
    if (id >= Tb * W) return;
    const int b = id / W, d = id - b * W + 1;
    PH[((size_t)(b / LC_NB) * W + (d - 1)) * LC_NB + (b % LC_NB)] = tw[(size_t)((b * d) & (My - 1)) * (Nt / My)];
}

// ---------------------------------------------------------------- stage 2
// grid = (np, 2W+1 [dv]); block 256.
// WM: compile-time bound on W (5, 10, 20) -- sized for MAX_L the accumulators took 228 registers (one CTA per SM, three waves)
template <int WM>
__global__ void __launch_bounds__(256) lagrow_kernel(const cplx *__restrict__ Q, int np, int W, int nsplit,
                                                    const double *__restrict__ bpart, int nchunk,
                                                    double *__restrict__ lag, Geom g, const cplx *__restrict__ tw) {
    const int p = blockIdx.x, dvi = blockIdx.y, Hx = g.Hx, Mx = g.Mx;
    double sc[WM + 1], sn[WM + 1];
#pragma unroll
    for (int d = 0; d <= WM; d++) { sc[d] = 0.0; sn[d] = 0.0; }
    for (int kx = threadIdx.x; kx <= Hx; kx += blockDim.x) {
        cplx q = mk(0, 0);
        for (int s = 0; s < nsplit; s++) q = cadd(q, Q[((size_t)(s * np + p) * (2 * W + 1) + dvi) * (Hx + 1) + kx]);
        const double gw = (kx == 0 || kx == Hx) ? 1.0 : 2.0;
        q.x *= gw; q.y *= gw;
        // exp(-2 pi i kx d/Mx) = e1^d from ONE coalesced table load: 2W+1 gathered loads per kx made this kernel
        // sector-request bound (55 us for a 38 MFLOP reduction); powers in a tree, at most 5 roundings deep
        const cplx e1 = tw[(size_t)(kx & (Mx - 1)) * (g.Nt / Mx)];
        cplx ep[WM + 1];
        ep[0] = mk(1.0, 0.0); ep[1] = e1;
#pragma unroll
        for (int d = 2; d <= WM; d++)
            if (d <= W) ep[d] = cmul(ep[d / 2], ep[d - d / 2]);
#pragma unroll
        for (int d = 0; d <= WM; d++)
            if (d <= W) { sc[d] = fma(q.x, ep[d].x, sc[d]); sn[d] = fma(q.y, -ep[d].y, sn[d]); } // cos = e.x, sin = -e.y
    }
    // one reduction for all 2(W+1) sums: shuffles inside a warp, then one pass through shared memory
    __shared__ double red[8][2 * (WM + 1)];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int d = 0; d <= WM; d++)
        if (d <= W) {
            double c = sc[d], sv = sn[d];
#pragma unroll
            for (int off = 16; off > 0; off >>= 1) { c += __shfl_down_sync(0xffffffffu, c, off); sv += __shfl_down_sync(0xffffffffu, sv, off); }
            if (lane == 0) { red[wid][2 * d] = c; red[wid][2 * d + 1] = sv; }
        }
    __syncthreads();
    const double scale = 1.0 / ((double)g.Mx * (double)g.My);
    const int nl = (2 * W + 1) * (2 * W + 1);
    if ((int)threadIdx.x <= W) {
        const int d = threadIdx.x;
        double c = 0.0, sv = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); k++) { c += red[k][2 * d]; sv += red[k][2 * d + 1]; }
        double vp = (c - sv) * scale, vm = (c + sv) * scale; // Re(q e^{+i th}), Re(q e^{-i th})
        const int ip = dvi * (2 * W + 1) + (W + d), im = dvi * (2 * W + 1) + (W - d);
        for (int k = 0; k < nchunk; k++) {
            vp += bpart[((size_t)k * np + p) * nl + ip];
            if (d > 0) vm += bpart[((size_t)k * np + p) * nl + im];
        }
        lag[(size_t)p * nl + ip] = vp;
        if (d > 0) lag[(size_t)p * nl + im] = vm;
    }
}

// lag[i] += sum over chunks of bpart[chunk][i]: the native-grid wrap corrections join the lag tables
__global__ void lagadd_kernel(double *__restrict__ lag, const double *__restrict__ bpart, int total, int nchunk) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= total) return;
    double v = lag[i];
    for (int k = 0; k < nchunk; k++) v += bpart[(size_t)k * total + i];
    lag[i] = v;
}

// ---------------------------------------------------------------- host side
// Launch shape of stage 1, fixed at plan creation (it sizes Q and the TMA boxes): 8 b-lanes per (pair, kx),
// KXC kx per CTA, pairs in even groups, CTAs of <= 192 threads so that two fit an SM with the accumulators in
// registers; the ring takes what two CTAs per SM leave of shared memory.
void lagcol_config(const Geom &g, int np, int ns, int W, LagCfg *c, size_t esz) {
    const int WB = W <= 3 ? 3 : W <= 5 ? 5 : W <= 6 ? 6 : W <= 10 ? 10 : 20;
    const int Tb = g.My / LC_NA;
    const int KXC = ns <= 7 ? 2 : 1;
    // wide form (lagcol_wide_kernel): all pairs in one CTA when that takes 193..384 threads and all lags fit one thread
    const bool wide = WB <= 10 && np * KXC * LC_NB > 192 && ((np * KXC + 3) & ~3) * LC_NB <= 384;
    int npg = (wide ? 384 : 192) / (LC_NB * KXC); if (npg > np) npg = np;
    int ngr = (np + npg - 1) / npg; npg = (np + ngr - 1) / ngr;   // even groups (21 pairs: 11 + 10)
    while ((npg * KXC) & 3) npg++;                                 // whole warps (inactive pair slots idle)
    const size_t stage = (size_t)ns * KXC * LC_NA * LC_NB * esz + (size_t)WB * LC_NB * sizeof(cplx); // the kernel folds WB lags (>= W)
    int nst = 4;
    while (nst > 2 && nst * stage > (size_t)110 * 1024) nst--;
    c->WB = WB; c->KXC = KXC; c->npg = npg; c->ngr = ngr; c->nkb = (g.Hx + 1 + KXC - 1) / KXC;
    c->halves = WB > 10 ? 2 : 1; c->wide = wide;
    int nsplit = 1;   // few kx blocks (small frames): split the ky range so that the machine still fills
    while ((long long)c->nkb * ngr * nsplit * c->halves < (wide ? 148 : 296) && Tb / (2 * nsplit) >= 2 * LC_NB) nsplit *= 2;
    c->nsplit = nsplit; c->rows_per_split = Tb / nsplit; c->nst = nst; c->smem = nst * stage;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// tensor map over spectra planes [plane][kx 0..Hx][a 0..15][b 0..Tb-1] (a complex = 2 doubles):
// box {8 b, 16 a, KXC kx, all planes}; rank 4 for the template set (NK planes, contiguous), rank 3 for one science spectrum
static cudaError_t make_lag_map(CUtensorMap *tm, const void *base, bool f32, int nplanes, int rank, int KXC, const Geom &g) {
    void *fn = nullptr; cudaDriverEntryPointQueryResult qr;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
    if (e != cudaSuccess) return e;
    if (!fn || qr != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
    const cuuint64_t Tb = (cuuint64_t)g.My / LC_NA;
    cuuint64_t dims[4] = {2 * Tb, LC_NA, (cuuint64_t)g.Hx + 1, (cuuint64_t)nplanes};
    const cuuint64_t eb = f32 ? 8 : 16; // bytes per complex element
    cuuint64_t strides[3] = {Tb * eb, (cuuint64_t)g.My * eb, ((cuuint64_t)g.Hx + 1) * g.My * eb};
    cuuint32_t box[4] = {2 * LC_NB, LC_NA, (cuuint32_t)KXC, (cuuint32_t)nplanes}, es[4] = {1, 1, 1, 1};
    CUresult r = ((EncodeTiledFn)fn)(tm, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, (cuuint32_t)rank, (void *)base, dims, strides, box, es,
                                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int WB> static cudaError_t lag_attr() {
    cudaError_t e = cudaFuncSetAttribute(lagcol_kernel<WB, cplx>, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(lagcol_kernel<WB, float2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024);
    if (WB <= 10) {
        constexpr int WW = WB <= 10 ? WB : 10;
        if (e == cudaSuccess) e = cudaFuncSetAttribute(lagcol_wide_kernel<WW, cplx>, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(lagcol_wide_kernel<WW, float2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024);
    }
    return e;
}

// plan creation (after the spectra are allocated): launch shapes, tensor maps, phase tables, kernel attributes
cudaError_t lags_init(sfft_plan *p) {
    const Geom &g = p->g;
    p->mapsO = new (std::nothrow) LagMaps(); p->mapsT = new (std::nothrow) LagMaps[NSCI]();
    if (!p->mapsO || !p->mapsT) return cudaErrorMemoryAllocation;
    cudaError_t e = make_lag_map(&p->mapsO->t, p->specT, p->spec32, g.NK, 4, p->cfgO.KXC, g);
    for (int n = 1; n <= NSCI && e == cudaSuccess; n++) {
        e = make_lag_map(&p->mapsT[n - 1].t, p->specT, p->spec32, g.NK, 4, p->cfgT[n - 1].KXC, g);
        for (int i = 0; i < n && e == cudaSuccess; i++) e = make_lag_map(&p->mapsT[n - 1].s[i], p->specSx[i], p->spec32, 1, 3, p->cfgT[n - 1].KXC, g);
    }
    if (e != cudaSuccess) return e;
    const int Tb = g.My / LC_NA;
    lag_phase_kernel<<<(Tb * p->cfgO.WB + 255) / 256, 256>>>(p->phO, p->cfgO.WB, g.My, p->tw, g.Nt);
    lag_phase_kernel<<<(Tb * p->cfgT[0].WB + 255) / 256, 256>>>(p->phT, p->cfgT[0].WB, g.My, p->tw, g.Nt);
    e = lag_attr<3>();
    if (e == cudaSuccess) e = lag_attr<5>();
    if (e == cudaSuccess) e = lag_attr<6>();
    if (e == cudaSuccess) e = lag_attr<10>();
    if (e == cudaSuccess) e = lag_attr<20>();
    return e;
}
void lags_free(sfft_plan *p) { delete p->mapsO; delete[] p->mapsT; p->mapsO = nullptr; p->mapsT = nullptr; }
size_t lag_q_elems(const sfft_plan *p) { // Q: the largest of the Omega pass and the Theta passes of 1..NSCI images
    const Geom &g = p->g;
    size_t q = (size_t)p->cfgO.nsplit * p->plO.np * (4 * g.w + 1) * (g.Hx + 1);
    for (int n = 1; n <= NSCI; n++) {
        const size_t qt = (size_t)p->cfgT[n - 1].nsplit * n * g.NK * g.L * (g.Hx + 1);
        if (qt > q) q = qt;
    }
    return q;
}

template <int WB>
static cudaError_t run_lagcol(sfft_plan *p, const LagMaps &maps, int ns, int nsci, const PairList &pl, int W, const LagCfg &c, bool science) {
    LagArgs la;
    la.ns = ns; la.nsci = nsci; la.npg = c.npg; la.KXC = c.KXC; la.W = W; la.nbs = c.rows_per_split; la.nst = c.nst; la.phW = c.WB; la.nkb = c.nkb;
    dim3 grid(c.ngr * c.halves, c.nkb, c.nsplit);
    if (science && p->factor_pending && !c.wide) {   // leave SMs to the factorisation running beside the pass (lagcol_kernel)
        const int per = c.ngr * c.halves * c.nsplit, cap = 2 * (p->sms - p->knob.factor_sms) / (per > 0 ? per : 1);
        if (cap >= 1 && cap < c.nkb) grid.y = cap;
    }
    KLaunch kl(p, science ? "lagcol_theta" : "lagcol_omega");
    constexpr int WW = WB <= 10 ? WB : 10;
    if (c.wide && p->spec32) lagcol_wide_kernel<WW, float2><<<grid, c.npg * c.KXC * LC_NB, c.smem, p->cur>>>(maps, la, pl, science ? p->phT : p->phO, p->Q, p->g);
    else if (c.wide) lagcol_wide_kernel<WW, cplx><<<grid, c.npg * c.KXC * LC_NB, c.smem, p->cur>>>(maps, la, pl, science ? p->phT : p->phO, p->Q, p->g);
    else if (p->spec32) lagcol_kernel<WB, float2><<<grid, c.npg * c.KXC * LC_NB, c.smem, p->cur>>>(maps, la, pl, science ? p->phT : p->phO, p->Q, p->g);
    else lagcol_kernel<WB, cplx><<<grid, c.npg * c.KXC * LC_NB, c.smem, p->cur>>>(maps, la, pl, science ? p->phT : p->phO, p->Q, p->g);
    return cudaGetLastError();
}

int border_chunks() { return 1; }

cudaError_t launch_lags(sfft_plan *p, const PairList &pl, int W, double *lag, bool science, int nsci) {
    const Geom &g = p->g;
    const LagCfg &c = science ? p->cfgT[nsci - 1] : p->cfgO;
    const LagMaps &maps = science ? p->mapsT[nsci - 1] : *p->mapsO;
    const int ns = science ? g.NK + nsci : g.NK;
    const int nsplit = c.nsplit;
    cudaError_t e;
    // side streams: the wrap corrections (independent of the column pass)
    int nchunk = 0;
    double *bpart = p->bpart;
    if (g.Mx != g.nx || g.My != g.ny) {
        nchunk = border_chunks();
        use_side(p, 1); // the caller forked already (template_side / science_side)
        if (W > 0 && science && nsci > 1) {
            // several science images: the wrap corrections image by image (their strips come from p->S), the pairs of
            // image i behind those of image i-1 in bpart (border_chunks() == 1)
            const int nl = (2 * W + 1) * (2 * W + 1);
            const double *keep = p->S;
            for (int i = 0; i < nsci; i++) {
                p->S = p->Sx[i];
                e = launch_border(p, p->plT, W, true, bpart + (size_t)i * g.NK * nl);
                if (e != cudaSuccess) { p->S = keep; return e; }
            }
            p->S = keep;
        } else if (W > 0) { e = launch_border(p, pl, W, science, bpart); if (e != cudaSuccess) return e; }
        else nchunk = 0;
    }
    back_to_main(p);
    if (c.WB == 3) e = run_lagcol<3>(p, maps, ns, science ? nsci : 0, pl, W, c, science);
    else if (c.WB == 5) e = run_lagcol<5>(p, maps, ns, science ? nsci : 0, pl, W, c, science);
    else if (c.WB == 6) e = run_lagcol<6>(p, maps, ns, science ? nsci : 0, pl, W, c, science);
    else if (c.WB == 10) e = run_lagcol<10>(p, maps, ns, science ? nsci : 0, pl, W, c, science);
    else e = run_lagcol<20>(p, maps, ns, science ? nsci : 0, pl, W, c, science);
    if (e != cudaSuccess) return e;
    {   // the row reduction does not wait for the wrap corrections (a chain of small kernels on a side stream that only gets
        // SMs once the column pass has ended -- 0.57 ms of it at L = 21): they are added afterwards (lagadd)
        KLaunch kl(p, science ? "lagrow_theta" : "lagrow_omega");
        const dim3 gr(pl.np, 2 * W + 1);
        if (W <= 5) lagrow_kernel<5><<<gr, 256, 0, p->cur>>>(p->Q, pl.np, W, nsplit, bpart, 0, lag, g, p->tw);
        else if (W <= 10) lagrow_kernel<10><<<gr, 256, 0, p->cur>>>(p->Q, pl.np, W, nsplit, bpart, 0, lag, g, p->tw);
        else lagrow_kernel<MAX_L - 1><<<gr, 256, 0, p->cur>>>(p->Q, pl.np, W, nsplit, bpart, 0, lag, g, p->tw);
    }
    join_side(p);
    if (nchunk > 0) {
        const int total = pl.np * (2 * W + 1) * (2 * W + 1);
        KLaunch kl(p, science ? "lagadd_theta" : "lagadd_omega");
        lagadd_kernel<<<(total + 255) / 256, 256, 0, p->cur>>>(lag, bpart, total, nchunk);
    }
    return cudaGetLastError();
}

} // namespace sfft
