// Host check of paper_2406_14542_b200/csrc/fft_reg.cuh (the register-tiled 4096-point FFT of the fused phi transform):
// the phase functions are __host__ __device__, so the 256 "threads" are run one after the other here, phase by phase
// (a device barrier separates the phases), and the result is compared with a direct O(N^2) DFT in long double, for
// both signs of the exponent.  Built and run by tests/test_fft_smem_cpu.py.
#include <cmath>
#include <complex>
#include <cstdio>
#include <vector>

#include "../paper_2406_14542_b200/csrc/fft_reg.cuh"
using namespace fftreg;

template <int SIGN>
double run() {
    const long double PI_L = 3.14159265358979323846264338327950288L;
    std::vector<double2> tw4096(256), tw256(16), s(HSMEM);
    for (int i = 0; i < 256; ++i) tw4096[i] = make_double2((double)cosl(-2 * PI_L * i / 4096), (double)sinl(-2 * PI_L * i / 4096));
    for (int i = 0; i < 16; ++i) tw256[i] = make_double2((double)cosl(-2 * PI_L * i / 256), (double)sinl(-2 * PI_L * i / 256));
    std::vector<std::complex<long double>> in(HLEN);
    unsigned long long st = 12345;
    auto rnd = [&]() { st = st * 6364136223846793005ULL + 1442695040888963407ULL; return (double)((st >> 11) * (1.0 / 9007199254740992.0)) - 0.5; };
    for (auto& v : in) v = {rnd(), rnd()};
    std::vector<double2> regs(HLEN);      // regs[t * 16 + j]: register j of thread t
    double2 x[16];
    for (int t = 0; t < HTHREADS; ++t) {
        for (int j = 0; j < 16; ++j) x[j] = make_double2((double)in[t + 256 * j].real(), (double)in[t + 256 * j].imag());
        phase_a<SIGN>(x, s.data(), t, tw4096.data());
    }
    for (int t = 0; t < HTHREADS; ++t) {
        phase_b1(x, s.data(), t);
        for (int j = 0; j < 16; ++j) regs[t * 16 + j] = x[j];
    }
    for (int t = 0; t < HTHREADS; ++t) {
        for (int j = 0; j < 16; ++j) x[j] = regs[t * 16 + j];
        phase_b2<SIGN>(x, s.data(), t, tw256.data());
    }
    double worst = 0.0, scale = 0.0;
    std::vector<std::complex<long double>> ref(HLEN);
    for (int q = 0; q < HLEN; ++q) {
        std::complex<long double> acc = 0;
        for (int i = 0; i < HLEN; ++i) {
            const long double ang = SIGN * 2 * PI_L * (long double)((long long)i * q % HLEN) / HLEN;
            acc += in[i] * std::complex<long double>(cosl(ang), sinl(ang));
        }
        ref[q] = acc;
        scale = std::max(scale, (double)std::abs(acc));
    }
    for (int t = 0; t < HTHREADS; ++t) {
        phase_c<SIGN>(x, s.data(), t);
        for (int c = 0; c < 16; ++c) {
            const double2 v = x[bitrev(c, 16)];
            const std::complex<long double> d = std::complex<long double>(v.x, v.y) - ref[t + 256 * c];
            worst = std::max(worst, (double)std::abs(d));
        }
    }
    printf("fft_reg 4096 sign %+d: max |err| / max |X| = %.3e\n", SIGN, worst / scale);
    return worst / scale;
}

int main() {
    const double e1 = run<-1>(), e2 = run<+1>();
    if (e1 > 5e-15 || e2 > 5e-15) {
        printf("FAILED\n");
        return 1;
    }
    printf("OK\n");
    return 0;
}
