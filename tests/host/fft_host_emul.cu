// Host emulation of the Stockham passes in csrc/sfft_fft.cuh: every "thread" j of one
// transform is run in turn, pass by pass, exactly as fft_block sequences them on the GPU,
// and the result is compared with a naive long-double DFT.  Prints "N dir max_rel_err".
// Built and run by tests/test_fft_host.py (CPU only; nvcc compiles it as host code).
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <vector>
#include "../../paper_2509_18544_b200/csrc/sfft_fft.cuh"
using namespace sfft;

template <int DIR> static double run(int log2N) {
    const int N = 1 << log2N, T = N >> 4, Nt = 8192;
    std::vector<cplx> tw(Nt), in(N), s(padded_len(N)), out(N);
    for (int k = 0; k < Nt; k++) { long double a = -2.0L * M_PIl * k / Nt; tw[k] = mk((double)cosl(a), (double)sinl(a)); }
    srand(1234 + log2N);
    for (int i = 0; i < N; i++) in[i] = mk(rand() / (double)RAND_MAX - 0.5, rand() / (double)RAND_MAX - 0.5);
    std::vector<cplx> regs((size_t)T * 16);
    for (int j = 0; j < T; j++) for (int q = 0; q < 16; q++) regs[(size_t)j * 16 + q] = in[j + q * T];
    int log2Ns = 0;
    for (int j = 0; j < T; j++) fft_pass<16, DIR, true>(&regs[(size_t)j * 16], s.data(), j, T, 0, tw.data(), Nt);
    for (int j = 0; j < T; j++) fft_load_canonical(&regs[(size_t)j * 16], s.data(), j, T);
    log2Ns = 4;
    while (log2Ns + 4 < log2N) {
        for (int j = 0; j < T; j++) fft_pass<16, DIR, true>(&regs[(size_t)j * 16], s.data(), j, T, log2Ns, tw.data(), Nt);
        for (int j = 0; j < T; j++) fft_load_canonical(&regs[(size_t)j * 16], s.data(), j, T);
        log2Ns += 4;
    }
    for (int j = 0; j < T; j++) {
        cplx *v = &regs[(size_t)j * 16];
        switch (log2N - log2Ns) {
        case 4: fft_pass<16, DIR, false>(v, s.data(), j, T, log2Ns, tw.data(), Nt); break;
        case 3: fft_pass<8, DIR, false>(v, s.data(), j, T, log2Ns, tw.data(), Nt); break;
        case 2: fft_pass<4, DIR, false>(v, s.data(), j, T, log2Ns, tw.data(), Nt); break;
        default: fft_pass<2, DIR, false>(v, s.data(), j, T, log2Ns, tw.data(), Nt); break;
        }
    }
    for (int j = 0; j < T; j++) for (int q = 0; q < 16; q++) out[j + q * T] = regs[(size_t)j * 16 + q];
    // naive DFT on a subset of outputs (all for small N)
    double maxerr = 0, maxv = 0;
    int step = N > 1024 ? 37 : 1;
    for (int k = 0; k < N; k += step) {
        long double re = 0, im = 0;
        for (int n = 0; n < N; n++) {
            long double a = DIR * 2.0L * M_PIl * (long double)(((long long)n * k) % N) / N;
            long double c = cosl(a), sn = sinl(a);
            re += in[n].x * c - in[n].y * sn; im += in[n].x * sn + in[n].y * c;
        }
        maxerr = fmax(maxerr, fmax(fabs(out[k].x - (double)re), fabs(out[k].y - (double)im)));
        maxv = fmax(maxv, fmax(fabs((double)re), fabs((double)im)));
    }
    return maxerr / maxv;
}

int main() {
    for (int l = 5; l <= 13; l++) {
        printf("%d -1 %.3e\n", 1 << l, run<-1>(l));
        printf("%d 1 %.3e\n", 1 << l, run<1>(l));
    }
    return 0;
}
