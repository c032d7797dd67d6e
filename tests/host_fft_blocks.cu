// Host-side check of the register FFT building blocks of paper_2605_28800_b200/csrc/fe_fft2.cuh (they are
// __host__ __device__): every recursion the kernels instantiate is compared with the O(N^2) definition of the DFT
// (PAPER.md:115 names the transform; Eq. 5-6 PAPER.md:66-72 is what it serves).  Compiled and run by
// tests/test_fft_blocks_host.py; prints one line "name N max_rel_error" per case.
#include "fe_fft2.cuh"
#include <cmath>
#include <complex>
#include <cstdio>
#include <vector>

using namespace fe::v2;
typedef std::complex<double> cd;

static std::vector<cd> signal(int n, bool upper_zero)
{
    std::vector<cd> x(n);
    for (int i = 0; i < n; ++i)
        x[i] = (upper_zero && i >= n / 2) ? cd(0, 0) : cd(std::sin(1.3 * i + 0.2) + 0.1 * i, std::cos(0.7 * i * i + 0.1));
    return x;
}
static cd dft(const std::vector<cd>& x, int k, int dir)
{
    const int n = (int)x.size();
    cd s = 0;
    for (int i = 0; i < n; ++i) s += x[i] * std::polar(1.0, dir * 2 * M_PI * (double)((long long)i * k % n) / n);
    return s;
}
template <typename T> static double report(const char* name, int n, const std::vector<cd>& x, const cx<T>* v, int dir,
                                           int nout, bool out_bitrev)
{
    double err = 0, nrm = 0;
    for (int k = 0; k < nout; ++k) {
        int p = k;
        if (out_bitrev) {
            p = 0;
            for (int b = 1, kk = k; b < n; b <<= 1, kk >>= 1) p = (p << 1) | (kk & 1);
        }
        const cd ref = dft(x, k, dir);
        err = std::fmax(err, std::abs(ref - cd(v[p].x, v[p].y)));
        nrm = std::fmax(nrm, std::abs(ref));
    }
    std::printf("%s %d %.3e\n", name, n, err / nrm);
    return err / nrm;
}

// DitF: v[p] = x[brev(p)] in, X[k] natural out
template <typename T, int N, int DIR, bool PIN, bool POUT> static void run_ditf(const char* name)
{
    const std::vector<cd> x = signal(N, PIN);
    cx<T> v[N];
    for (int p = 0; p < N; ++p) {
        const int n = brev<N>(p);
        // positions the pruned transform must not read are poisoned
        v[p] = (PIN && (p & 1)) ? cx<T>{(T)1e30, (T)1e30} : cx<T>{(T)x[n].real(), (T)x[n].imag()};
    }
    DitF<T, DIR, N, 0, PIN, POUT>::run(v);
    report<T>(name, N, x, v, DIR, POUT ? N / 2 : N, false);
}
// Dif: natural in, v[p] = X[brev(p)] out
template <typename T, int N, int DIR, bool PRUNE> static void run_dif(const char* name)
{
    const std::vector<cd> x = signal(N, PRUNE);
    cx<T> v[N];
    for (int n = 0; n < N; ++n) v[n] = (PRUNE && n >= N / 2) ? cx<T>{(T)1e30, (T)1e30} : cx<T>{(T)x[n].real(), (T)x[n].imag()};
    Dif<T, DIR, N, 0, PRUNE>::run(v);
    report<T>(name, N, x, v, DIR, N, true);
}
// Dit: v[p] = x[brev(p)] in, natural out
template <typename T, int N, int DIR> static void run_dit(const char* name)
{
    const std::vector<cd> x = signal(N, false);
    cx<T> v[N];
    for (int p = 0; p < N; ++p) v[p] = cx<T>{(T)x[brev<N>(p)].real(), (T)x[brev<N>(p)].imag()};
    Dit<T, DIR, N>::run(v);
    report<T>(name, N, x, v, DIR, N, false);
}

int main()
{
    run_ditf<double, 32, -1, false, false>("ditf_fwd");
    run_ditf<double, 32, -1, true, false>("ditf_fwd_pin");
    run_ditf<double, 32, +1, false, true>("ditf_inv_pout");
    run_ditf<double, 32, +1, false, false>("ditf_inv");
    run_ditf<double, 16, -1, false, false>("ditf_fwd");
    run_ditf<double, 16, -1, true, false>("ditf_fwd_pin");
    run_ditf<double, 16, +1, false, true>("ditf_inv_pout");
    run_ditf<double, 8, -1, false, false>("ditf_fwd");
    run_ditf<double, 8, +1, false, false>("ditf_inv");
    run_ditf<double, 8, -1, true, false>("ditf_fwd_pin");
    run_ditf<double, 4, +1, false, true>("ditf_inv_pout");
    run_ditf<double, 2, -1, false, false>("ditf_fwd");
    run_dif<double, 32, -1, false>("dif_fwd");
    run_dif<double, 32, -1, true>("dif_fwd_prune");
    run_dif<double, 32, +1, false>("dif_inv");
    run_dif<double, 16, -1, true>("dif_fwd_prune");
    run_dif<double, 16, +1, false>("dif_inv");
    run_dif<double, 8, -1, false>("dif_fwd");
    run_dif<double, 8, +1, false>("dif_inv");
    run_dif<double, 4, -1, true>("dif_fwd_prune");
    run_dit<double, 32, +1>("dit_inv");
    run_dit<double, 16, -1>("dit_fwd");
    run_dit<double, 8, +1>("dit_inv");
    run_ditf<float, 32, -1, true, false>("f32_ditf_fwd_pin");
    run_ditf<float, 32, +1, false, true>("f32_ditf_inv_pout");
    run_dif<float, 16, -1, false>("f32_dif_fwd");
    return 0;
}
