// Host check of paper_2406_14542_b200/csrc/fft_smem.cuh (the shared-memory FFT of the fused theta chains):
// the stage functions are __host__ __device__, so the "threads" are run one after the other here and the
// result is compared with a direct O(N^2) DFT in long double.  Checks, for every supported N: the forward
// chain (fused radix-2 stage + stages + register-resident last stage) against the DFT at the
// digit-reversed positions freq_of_pos gives, and the inverse chain (first stage from registers +
// stages + fused radix-2) as its exact inverse.  Built and run by tests/test_fft_smem_cpu.py.
#include <cmath>
#include <complex>
#include <cstdio>
#include <vector>

#include "../paper_2406_14542_b200/csrc/fft_smem.cuh"
using namespace fftsm;

template <int N, int SIGN>
struct HostExec {
    double2* s;
    const double2* stw;
    int T;
    template <int R, int NS>
    void dif() {
        for (int t = 0; t < T; ++t) stage_dif<N, R, NS, SIGN>(s, t, T, stw + stage_table_offset(N, NS));
    }
    template <int R, int NS>
    void dit() {
        for (int t = 0; t < T; ++t) stage_dit<N, R, NS, SIGN>(s, t, T, stw + stage_table_offset(N, NS));
    }
};

template <int N>
int run() {
    constexpr int T = N >= 512 ? N / 16 : 32, E = N / T, RL = last_radix(N / 2);
    const long double PI_L = 3.14159265358979323846264338327950288L;
    std::vector<double2> tw2(N / 2), stw(stage_table_len(N) + 1), s(padded_len(N));
    for (int i = 0; i < N / 2; ++i) tw2[i] = make_double2((double)cosl(-2 * PI_L * i / N), (double)sinl(-2 * PI_L * i / N));
    {
        size_t o = 0;
        for (int ns = N / 2; ns >= 32; ns /= 16)
            for (int i = 0; i < ns / 16; ++i)
                stw[o++] = make_double2((double)cosl(-2 * PI_L * i / ns), (double)sinl(-2 * PI_L * i / ns));
    }
    std::vector<std::complex<double>> x(N), X(N);
    unsigned long long st = 88172645463325252ULL + N;
    auto rnd = [&]() { st ^= st << 13; st ^= st >> 7; st ^= st << 17; return (double)(st >> 11) / 9007199254740992.0 - 0.5; };
    for (auto& v : x) v = {rnd(), rnd()};
    for (int q = 0; q < N; ++q) {
        std::complex<long double> a = 0;
        for (int r = 0; r < N; ++r) {
            const long double ang = -2 * PI_L * (long double)(((long long)q * r) % N) / N;
            a += std::complex<long double>(x[r]) * std::complex<long double>(cosl(ang), sinl(ang));
        }
        X[q] = std::complex<double>((double)a.real(), (double)a.imag());
    }
    // forward
    for (int i = 0; i < N / 2; ++i) {
        const double2 a = make_double2(x[i].real(), x[i].imag()), b = make_double2(x[i + N / 2].real(), x[i + N / 2].imag());
        s[pad(i)] = make_double2(a.x + b.x, a.y + b.y);
        s[pad(i + N / 2)] = cmul(make_double2(a.x - b.x, a.y - b.y), tw2[i]);
    }
    HostExec<N, -1> f{s.data(), stw.data(), T};
    forward_stages<N / 2>(f);
    std::vector<double2> regs((size_t)T * E);
    double err = 0, nrm = 0;
    for (int t = 0; t < T; ++t) {
        double2 c[E];
        last_stage_to_regs<N, RL, -1, E>(s.data(), t, T, c);
        for (int e = 0; e < E; ++e) {
            const int pos = RL * (t + T * (e / RL)) + e % RL, q = freq_of_pos<N>(pos);
            err += std::norm(std::complex<double>(c[e].x, c[e].y) - X[q]);
            nrm += std::norm(X[q]);
            regs[(size_t)t * E + e] = c[e];
        }
    }
    const double e_fwd = std::sqrt(err / nrm);
    // inverse
    for (int t = 0; t < T; ++t) {
        double2 c[E];
        for (int e = 0; e < E; ++e) c[e] = regs[(size_t)t * E + e];
        first_stage_from_regs<N, RL, +1, E>(s.data(), t, T, c);
    }
    HostExec<N, +1> g{s.data(), stw.data(), T};
    inverse_stages<N / 2>(g);
    err = nrm = 0;
    for (int i = 0; i < N / 2; ++i) {
        const double2 z0 = s[pad(i)], z1 = cmul(s[pad(i + N / 2)], cconj(tw2[i]));
        const std::complex<double> o0(z0.x + z1.x, z0.y + z1.y), o1(z0.x - z1.x, z0.y - z1.y);
        err += std::norm(o0 / (double)N - x[i]) + std::norm(o1 / (double)N - x[i + N / 2]);
        nrm += std::norm(x[i]) + std::norm(x[i + N / 2]);
    }
    const double e_inv = std::sqrt(err / nrm);
    std::printf("N=%d forward %.3e roundtrip %.3e\n", N, e_fwd, e_inv);
    return (e_fwd < 5e-15 && e_inv < 5e-15) ? 0 : 1;
}

int main() {
    int bad = 0;
    bad += run<128>();
    bad += run<256>();
    bad += run<512>();
    bad += run<1024>();
    bad += run<2048>();
    bad += run<4096>();
    bad += run<8192>();
    std::printf(bad ? "FAIL\n" : "OK\n");
    return bad;
}
