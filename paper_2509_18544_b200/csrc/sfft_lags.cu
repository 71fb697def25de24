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
//   lagcol_kernel  stage 1: Q[p][dv][kx] = sum_ky conj(A)B e^{2 pi i ky dv/My}, thread = (pair, kx),
//                  rows streamed through a cp.async shared-memory pipeline shared by all pairs
//   lagedge_kernel the packed column kx = 0 (DC + i Nyquist) untangled -> Q[.][.][0], Q[.][.][Hx]
//   (sfft_border.cu) the wrap corrections X_N - X_M from border strips
//   lagrow_kernel  stage 2: lag[p][dv][du] = 1/(Mx My) sum_kx g Re(Q e^{2 pi i kx du/Mx}) + border
#include <cstdio>
#include <cstdlib>
#include "sfft_internal.h"

namespace sfft {

struct SpecSet { const cplx *p[MAX_NP + NSCI]; };

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
    unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gsrc));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

// mbarrier helpers (shared::cta): the lag pipeline synchronises per STAGE (copies landed / stage consumed)
// instead of with CTA-wide barriers, so warps may run up to a stage apart
__device__ __forceinline__ void mbar_init(unsigned long long *b, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(b)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *b) {
    asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"((unsigned)__cvta_generic_to_shared(b)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_on_copies(unsigned long long *b) { // arrives when this thread's earlier cp.async land
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"((unsigned)__cvta_generic_to_shared(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *b, unsigned parity) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(b);
    asm volatile("{\n.reg .pred p;\nWAIT_%=:\nmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}\n" ::"r"(a), "r"(parity) : "memory");
}

constexpr int LC_NA = 16;  // decimation factor: ky = b + (My/16) a, a = 0..15
constexpr int LC_NST = 4;  // cp.async pipeline stages (prefetch distance 2, refill of the stage consumed 2 steps ago)

// Stage 1, output-pruned inverse DFT along ky by decimation:
//   Q[dv] = sum_ky P[ky] e^{2 pi i ky dv/My},  P = conj(A) B,  ky = b + Tb a  (Tb = My/16)
//         = sum_b e^{2 pi i b dv/My} F_b[dv mod 16],   F_b[m] = sum_a P[b + Tb a] e^{2 pi i a m/16}.
// A thread owns (pair, kx): per b it forms the 16 products, runs one register-resident 16-point DFT
// and folds the outputs it needs (DLO <= dv <= DHI) into its accumulators with one complex
// multiply-add each: ~19 FP64 instructions per spectrum element and pair instead of 4 + 4(2W+1)/2... of the
// direct sum.  The rows {b + Tb a} of all spectra of the CTA's kx chunk and the W phase factors of b
// arrive through a cp.async shared-memory pipeline shared by all pairs.
// grid = (kx blocks, pair groups, b splits * halves); block = npg * KXC threads.
// dynamic smem: LC_NST * (16 * ns * KXC + WB) cplx
template <int DLO, int DHI>
__device__ __forceinline__ void lag_fold(const cplx *x, const cplx *ph, cplx *acc) {
#pragma unroll
    for (int d = DLO; d <= DHI; d++) {
        const cplx v = x[((d % 16) + 16) % 16];
        cplx &a = acc[d - DLO];
        if (d == 0) { a.x += v.x; a.y += v.y; }
        else {
            const cplx e = ph[(d > 0 ? d : -d) - 1];       // exp(-i phi |d|): cos = e.x, sin = -e.y
            const double c = e.x, sn = d > 0 ? -e.y : e.y;  // multiply by exp(+i phi d)
            a.x = fma(v.x, c, a.x); a.x = fma(-v.y, sn, a.x);
            a.y = fma(v.x, sn, a.y); a.y = fma(v.y, c, a.y);
        }
    }
}

template <int DLO, int DHI, int WB>
__device__ __forceinline__ void lagcol_body(const SpecSet &ss, int ns, const PairList &pl, int npg, int KXC, int W, int nbs,
                                            int zsplit, cplx *__restrict__ Q, const Geom &g, const cplx *__restrict__ tw,
                                            cplx *tile) {
    const int Hx = g.Hx, My = g.My, Tb = My / LC_NA;
    const int row_elems = ns * KXC, stage_elems = LC_NA * row_elems + WB;
    const int kx0 = blockIdx.x * KXC;
    const int pl0 = blockIdx.y * npg;
    const int b0 = zsplit * nbs, b1 = min(Tb, b0 + nbs);
    const int nIt = max(0, b1 - b0);
    const int lp = threadIdx.x / KXC, lane = threadIdx.x - lp * KXC;
    const int p = pl0 + lp;
    const bool active = (p < pl.np) && (lp < npg);
    const int sa = active ? pl.a[p] : 0, sb = active ? pl.b[p] : 0;
    const int twsy = g.Nt / My;
    constexpr int NACC = DHI - DLO + 1;
    cplx acc[NACC];
#pragma unroll
    for (int d = 0; d < NACC; d++) acc[d] = mk(0.0, 0.0);

    // division-free tile copy: a thread copies the same (spectrum, kx) column slots of every stage
    // (row_elems <= 2 blockDim: np >= ns - 1), 16 rows each, plus one phase factor
    const cplx *gsrc[2]; int soff[2];
#pragma unroll
    for (int u = 0; u < 2; u++) {
        const int idx = threadIdx.x + u * blockDim.x;
        gsrc[u] = nullptr; soff[u] = 0;
        if (idx < row_elems) {
            const int s = idx / KXC; int kx = kx0 + (idx - s * KXC); if (kx >= Hx) kx = Hx - 1;
            gsrc[u] = ss.p[s] + spec_idx(0, kx, My); soff[u] = idx;
        }
    }
    const size_t astride = (size_t)Tb * 2; // tile-major spectra: consecutive ky of one column are 2 elements apart
    auto issue = [&](int it) {
        if (it < nIt) {
            cplx *st = tile + (size_t)(it % LC_NST) * stage_elems;
            const int b = b0 + it;
#pragma unroll
            for (int u = 0; u < 2; u++)
                if (gsrc[u]) {
                    const cplx *src = gsrc[u] + (size_t)b * 2;
#pragma unroll
                    for (int a = 0; a < LC_NA; a++) cp_async16(st + a * row_elems + soff[u], src + a * astride);
                }
            for (int d = threadIdx.x; d < WB; d += blockDim.x)
                cp_async16(st + LC_NA * row_elems + d, tw + (size_t)((b * (d + 1)) & (My - 1)) * twsy);
        }
        cp_async_commit();
    };

    // per-stage mbarriers: full[s] completes when every thread's copies of the stage have landed, done[s] when every
    // thread has consumed it.  A stage is refilled two steps after its use, so both waits are normally already satisfied.
    __shared__ unsigned long long full[LC_NST], done[LC_NST];
    if (threadIdx.x == 0)
        for (int k = 0; k < LC_NST; k++) { mbar_init(&full[k], blockDim.x); mbar_init(&done[k], blockDim.x); }
    __syncthreads();
    for (int it = 0; it < 2; it++)
        if (it < nIt) { issue(it); mbar_arrive_on_copies(&full[it]); }
    for (int it = 0; it < nIt; it++) {
        const int st_i = it % LC_NST;
        mbar_wait(&full[st_i], (unsigned)(it / LC_NST) & 1u);
        if (it + 2 < nIt) {
            const int sr = (it + 2) % LC_NST;
            if (it >= 2) mbar_wait(&done[sr], (unsigned)((it - 2) / LC_NST) & 1u);
            issue(it + 2);
            mbar_arrive_on_copies(&full[sr]);
        }
        if (active) {
            const cplx *st = tile + (size_t)st_i * stage_elems;
            cplx x[LC_NA];
#pragma unroll
            for (int a = 0; a < LC_NA; a++) {
                const cplx A = st[a * row_elems + sa * KXC + lane], B = st[a * row_elems + sb * KXC + lane];
                x[a] = cmulc(A, B);
            }
            dft16<1>(x);
            lag_fold<DLO, DHI>(x, st + LC_NA * row_elems, acc);
        }
        mbar_arrive(&done[st_i]);
    }
    const int kx = kx0 + lane;
    if (active && kx < Hx && kx > 0) { // kx = 0 is the packed column: lagedge_kernel owns Q[.][.][0]
        cplx *q = Q + ((size_t)(zsplit * pl.np + p) * (2 * W + 1)) * (Hx + 1) + kx;
#pragma unroll
        for (int d = DLO; d <= DHI; d++)
            if (d >= -W && d <= W) q[(size_t)(W + d) * (Hx + 1)] = acc[d - DLO];
    }
}

// WB <= 10: one thread folds all 2 WB + 1 lags.  WB = 20: the lag range is split in two halves
// (blockIdx.z parity) to keep the accumulators in registers; both halves write disjoint rows of Q.
template <int WB>
__global__ void __launch_bounds__(192, WB > 10 ? 1 : 2)
lagcol_kernel(SpecSet ss, int ns, PairList pl, int npg, int KXC, int W, int nbs, cplx *__restrict__ Q, Geom g,
              const cplx *__restrict__ tw) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    cplx *tile = reinterpret_cast<cplx *>(smem_raw);
    if (WB > 10) {
        const int half = blockIdx.z & 1, zs = blockIdx.z >> 1;
        if (half == 0) lagcol_body<0, WB, WB>(ss, ns, pl, npg, KXC, W, nbs, zs, Q, g, tw, tile);
        else lagcol_body<-WB, -1, WB>(ss, ns, pl, npg, KXC, W, nbs, zs, Q, g, tw, tile);
    } else {
        lagcol_body<-WB, WB, WB>(ss, ns, pl, npg, KXC, W, nbs, blockIdx.z, Q, g, tw, tile);
    }
}

// deterministic block sum of one double per thread (blockDim.x <= 1024, power of two)
__device__ __forceinline__ double block_sum(double v, double *sh) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    __syncthreads();
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    double r = 0.0;
    if (threadIdx.x == 0) for (int k = 0; k < (int)(blockDim.x >> 5); k++) r += sh[k];
    return r; // valid in thread 0
}

// grid = (np, 2W+1); block 256.  Column 0 holds F = F0 + i FH (F0, FH: column spectra of the real
// columns kx = 0 and kx = Hx of the row transform): F0[ky] = (F[ky] + conj F[-ky])/2,
// FH[ky] = (F[ky] - conj F[-ky])/(2i).
__global__ void __launch_bounds__(256) lagedge_kernel(SpecSet ss, PairList pl, int W, int nsplit, cplx *__restrict__ Q,
                                                     Geom g, const cplx *__restrict__ tw) {
    __shared__ double sh[32];
    const int p = blockIdx.x, dv = (int)blockIdx.y - W;
    const int Hx = g.Hx, My = g.My;
    const cplx *FA = ss.p[pl.a[p]], *FB = ss.p[pl.b[p]];
    double q0r = 0, q0i = 0, qhr = 0, qhi = 0;
    for (int ky = threadIdx.x; ky < My; ky += blockDim.x) {
        const int kn = (My - ky) & (My - 1);
        const cplx a = FA[(size_t)ky * 2], am = cconj(FA[(size_t)kn * 2]); // column 0 of tile 0
        const cplx b = FB[(size_t)ky * 2], bm = cconj(FB[(size_t)kn * 2]);
        const cplx A0 = mk(0.5 * (a.x + am.x), 0.5 * (a.y + am.y)), AH = mk(0.5 * (a.y - am.y), -0.5 * (a.x - am.x));
        const cplx B0 = mk(0.5 * (b.x + bm.x), 0.5 * (b.y + bm.y)), BH = mk(0.5 * (b.y - bm.y), -0.5 * (b.x - bm.x));
        cplx e = tw[(size_t)((ky * (dv + My)) & (My - 1)) * (g.Nt / My)];
        e.y = -e.y; // exp(+2 pi i ky dv/My)
        const cplx P0 = cmul(cmulc(A0, B0), e), PH = cmul(cmulc(AH, BH), e);
        q0r += P0.x; q0i += P0.y; qhr += PH.x; qhi += PH.y;
    }
    q0r = block_sum(q0r, sh); q0i = block_sum(q0i, sh); qhr = block_sum(qhr, sh); qhi = block_sum(qhi, sh);
    if (threadIdx.x == 0)
        for (int s = 0; s < nsplit; s++) {
            cplx *q = Q + ((size_t)(s * pl.np + p) * (2 * W + 1) + blockIdx.y) * (Hx + 1);
            q[0] = s == 0 ? mk(q0r, q0i) : mk(0, 0);
            q[Hx] = s == 0 ? mk(qhr, qhi) : mk(0, 0);
        }
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

// ---------------------------------------------------------------- host side
// Launch shape of stage 1 (also used by the plan to size Q): pick the kx chunk and the b split that
// minimise  waves * (work per CTA)  on 148 SMs x CTAs per SM, preferring wide chunks and few splits.
// min_split > 1: cut the ky range into at least that many CTAs per kx chunk -- short-lived CTAs, so that the
// kernels of a factorisation running beside this pass find free SM slots often (see sfft_build_system).
// reserve > 0: leave that many CTA slots free (a factorisation running beside this pass then finds room)
void lagcol_config(const Geom &g, int np, int ns, int W, LagCfg *c, int min_split, int reserve) {
    const int WB = W <= 3 ? 3 : W <= 5 ? 5 : W <= 6 ? 6 : W <= 10 ? 10 : 20;
    const int halves = WB > 10 ? 2 : 1, per_sm = WB > 10 ? 1 : 2, maxthreads = 192;
    const int Tb = g.My / LC_NA;
    double best = 1e300; int bK = 4, bS = 1, bG = np;
    // A science-side pass that shares the machine with a factorisation (reserve > 0): measured at 4088^2, L = 11, DK = 2,
    // CTAs of about 64 threads (410 x 60 threads) beat the 256 x 96 threads the cost model below prefers by 0.11 ms per
    // step -- the pass itself is shorter (0.30 vs 0.38 ms) and the factorisation's small kernels find room on every SM
    // (0.52 vs 0.66 ms); the landscape is rugged (KXC = 8 and 12 are both worse), so the rule is empirical:
    // the widest even chunk with npg * KXC <= 64.
    int kfix = 0;
    if (reserve > 0 && per_sm == 2 && np <= 32) { kfix = (64 / np) & ~1; if (kfix > 32) kfix = 32; if (kfix < 4) kfix = 0; }
    for (int KXC = 4; KXC <= 32; KXC++) {
        if (KXC > g.Hx) break;
        if (kfix && kfix <= g.Hx && KXC != kfix) continue;
        if ((size_t)LC_NST * (LC_NA * ns * KXC + WB) * sizeof(cplx) > (size_t)(per_sm == 2 ? 113 : 200) * 1024) break;
        int npg = maxthreads / KXC; if (npg > np) npg = np; if (npg < 1) continue;
        const int ngr = (np + npg - 1) / npg, nkb = (g.Hx + KXC - 1) / KXC;
        for (int nsplit = 1; nsplit <= 16; nsplit *= 2) {
            if (Tb / nsplit < 4 && nsplit > 1) break;
            if (nsplit < min_split && Tb / (2 * nsplit) >= 4 && nsplit < 16) continue;
            const long long ncta = (long long)nkb * ngr * nsplit * halves;
            long long slots = 148LL * per_sm;
            if (reserve > 0 && slots > 4 * reserve) slots -= reserve;
            if (kfix && ncta < slots && Tb / (2 * nsplit) >= 4 && nsplit < 16) continue; // small CTAs: at least one per slot
            const long long waves = (ncta + slots - 1) / slots;
            // a CTA with few threads keeps the FP64 pipes idle: charge it as if it had at least 160
            const int thr = npg * KXC < 160 ? 160 : npg * KXC;
            double cost = (double)waves * thr * ((Tb + nsplit - 1) / nsplit + 6);
            cost *= 1.0 + 0.01 * nsplit + (KXC < 8 ? 0.03 * (8 - KXC) : 0.0);
            if (KXC & 1) cost *= 1.2; // tile-major spectra: an odd chunk splits 32-byte sectors; and a grid that leaves a few
                                      // CTA slots free lets the small side-stream kernels run beside this pass
            if (cost < best) { best = cost; bK = KXC; bS = nsplit; bG = npg; }
        }
    }
    // Template pass with all pairs in ONE group and fewer CTAs than slots (21 pairs, L = 11: 256 CTAs x 168 threads on 296
    // slots -- 40 SMs get one CTA, the others two): the next narrower even chunk in two ky-splits deals out evenly
    // (684 CTAs x 126 threads, 4-5 per SM).  Measured: 0.420 -> 0.392 ms for the column kernel, 0.495 -> 0.458 ms for the
    // stage; 342 x 126 (no split) 0.457 ms, 1024 x 84 (KXC 4) 0.43 ms, 512 x 168 0.418 ms.  Only this shape is evidenced.
    if (np >= ns && np >= 16 && per_sm == 2 && bS == 1 && bG == np && bK >= 8 && !(bK & 1) && min_split <= 1 &&
        (long long)((g.Hx + bK - 1) / bK) < 148LL * per_sm && Tb >= 16) {
        bK -= 2; bS = 2;
    }
    if (const char *e = getenv(np < ns ? "SFFT_LAG_KXC_SCI" : "SFFT_LAG_KXC")) { // experiment knob: force the chunk width; pairs split evenly over the groups
        const int k = atoi(e);
        if (k >= 2 && k <= 32 && k <= g.Hx) { bK = k; bG = maxthreads / k < np ? maxthreads / k : np; }
    }
    { const int ngr0 = (np + bG - 1) / bG; bG = (np + ngr0 - 1) / ngr0; } // even pair groups (21 pairs in 2 groups: 11 + 10, not 13 + 8)
    c->WB = WB; c->KXC = bK; c->npg = bG; c->nkb = (g.Hx + bK - 1) / bK; c->ngr = (np + bG - 1) / bG;
    c->nsplit = bS; c->halves = halves;
    c->rows_per_split = (Tb + bS - 1) / bS; // in units of b
}

template <int WB>
static cudaError_t run_lagcol(sfft_plan *p, const SpecSet &ss, int ns, const PairList &pl, int W, const LagCfg &c, bool science) {
    const Geom &g = p->g;
    const size_t smem = (size_t)LC_NST * (LC_NA * ns * c.KXC + WB) * sizeof(cplx);
    cudaError_t e = cudaFuncSetAttribute(lagcol_kernel<WB>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (e != cudaSuccess) return e;
    dim3 grid(c.nkb, c.ngr, c.nsplit * c.halves);
    { KLaunch kl(p, science ? "lagcol_theta" : "lagcol_omega"); lagcol_kernel<WB><<<grid, c.npg * c.KXC, smem, p->cur>>>(ss, ns, pl, c.npg, c.KXC, W, c.rows_per_split, p->Q, g, p->tw); }
    return cudaGetLastError();
}

int border_chunks() { return 1; }
int theta_reserve() { static int v = -1; if (v < 0) { const char *e = getenv("SFFT_THETA_RESERVE"); v = e ? atoi(e) : 40; } return v; }
int theta_min_split() { static int v = -1; if (v < 0) { const char *e = getenv("SFFT_THETA_SPLIT"); v = e ? atoi(e) : 1; } return v; }

cudaError_t launch_lags(sfft_plan *p, const PairList &pl, int W, double *lag, bool science, int nsci) {
    const Geom &g = p->g;
    SpecSet ss;
    for (int t = 0; t < g.NK; t++) ss.p[t] = p->specT + (size_t)t * g.My * g.Hx;
    for (int i = 0; i < NSCI; i++) ss.p[g.NK + i] = (i < nsci && i > 0) ? p->specSx[i] : p->specS;
    const int ns = science ? g.NK + nsci : g.NK;
    static int omega_split = -1; // SFFT_OMEGA_SPLIT=8 shortens the column kernel by 8 % but lengthens the stage (side-stream kernels wait, more partials)
    if (omega_split < 0) { const char *e = getenv("SFFT_OMEGA_SPLIT"); omega_split = e ? atoi(e) : 1; }
    LagCfg c; lagcol_config(g, pl.np, ns, W, &c, science ? theta_min_split() : omega_split, science && p->factor_pending && pl.np >= 6 ? theta_reserve() : 0); // DK <= 1: the factor is short, the plain config is 4 % faster
    const int nsplit = c.nsplit;
    if (getenv("SFFT_VERBOSE")) fprintf(stderr, "lagcfg sci=%d np=%d WB=%d KXC=%d npg=%d nkb=%d ngr=%d nsplit=%d halves=%d threads=%d ctas=%d\n", (int)science, pl.np, c.WB, c.KXC, c.npg, c.nkb, c.ngr, c.nsplit, c.halves, c.npg * c.KXC, c.nkb * c.ngr * c.nsplit * c.halves);
    cudaError_t e;
    // side stream: the packed column kx = 0 / Hx and the wrap corrections (independent of the column pass)
    use_side(p, 0); // the caller forked already (template_side / science_side)
    { KLaunch kl(p, science ? "lagedge_theta" : "lagedge_omega"); lagedge_kernel<<<dim3(pl.np, 2 * W + 1), 256, 0, p->cur>>>(ss, pl, W, nsplit, p->Q, g, p->tw); }
    int nchunk = 0;
    double *bpart = p->bpart;
    if (g.Mx != g.nx || g.My != g.ny) {
        nchunk = border_chunks();
        use_side(p, 1);
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
    if (c.WB == 3) e = run_lagcol<3>(p, ss, ns, pl, W, c, science);
    else if (c.WB == 5) e = run_lagcol<5>(p, ss, ns, pl, W, c, science);
    else if (c.WB == 6) e = run_lagcol<6>(p, ss, ns, pl, W, c, science);
    else if (c.WB == 10) e = run_lagcol<10>(p, ss, ns, pl, W, c, science);
    else e = run_lagcol<20>(p, ss, ns, pl, W, c, science);
    if (e != cudaSuccess) return e;
    join_side(p);
    {
        KLaunch kl(p, science ? "lagrow_theta" : "lagrow_omega");
        const dim3 gr(pl.np, 2 * W + 1);
        if (W <= 5) lagrow_kernel<5><<<gr, 256, 0, p->cur>>>(p->Q, pl.np, W, nsplit, bpart, nchunk, lag, g, p->tw);
        else if (W <= 10) lagrow_kernel<10><<<gr, 256, 0, p->cur>>>(p->Q, pl.np, W, nsplit, bpart, nchunk, lag, g, p->tw);
        else lagrow_kernel<MAX_L - 1><<<gr, 256, 0, p->cur>>>(p->Q, pl.np, W, nsplit, bpart, nchunk, lag, g, p->tw);
    }
    return cudaGetLastError();
}

} // namespace sfft
