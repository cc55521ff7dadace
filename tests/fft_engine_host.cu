// Host-side emulation of csrc/fft.cuh: the CTA's threads are loops, __syncthreads() is the loop boundary.
// Checks the butterflies, the Stockham index logic, the pass schedule and the shared-memory padding against a
// direct O(N^2) DFT in fp64.  Built and run by tests/test_fft_engine_host.py (no GPU needed).
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "../paper_2203_02479_b200/csrc/fft.cuh"

using namespace wcsim;

template <int N, int C, int E, int DIR, int P, bool R32 = false>
static void emulate(std::vector<float2> &regs, std::vector<float2> &smem, const float2 *tw)
{
    constexpr int NT = (N / E) * C;
    constexpr int R = PassRadix<N, P, R32>::value;
    constexpr int SH = R32 ? 5 : 4;
    for (int t = 0; t < NT; ++t) {
        float2(&v)[E] = *reinterpret_cast<float2(*)[E]>(&regs[(size_t)t * E]);
        fft_pass<N, E, R, P, DIR>(v, t / C, tw);
    }
    if constexpr (P * R < N) {
        for (auto &s : smem) s = make_float2(NAN, NAN);
        for (int t = 0; t < NT; ++t) {
            float2(&v)[E] = *reinterpret_cast<float2(*)[E]>(&regs[(size_t)t * E]);
            fft_store<N, C, E, R, P, SH>(v, smem.data(), t / C, t % C);
        }
        for (int t = 0; t < NT; ++t) {
            float2(&v)[E] = *reinterpret_cast<float2(*)[E]>(&regs[(size_t)t * E]);
            fft_load<N, C, E, SH>(v, smem.data(), t / C, t % C);
        }
        emulate<N, C, E, DIR, P * R, R32>(regs, smem, tw);
    }
}

template <int N, int C, int E, int DIR, bool R32 = false>
static double check()
{
    constexpr int NT = (N / E) * C;
    std::vector<float2> tw(tw_size(N));
    build_pass_twiddles(N, tw.data());
    std::vector<double> xr((size_t)N * C), xi((size_t)N * C);
    srand(N * 31 + C * 7 + E + DIR);
    for (auto &x : xr) x = rand() / (double)RAND_MAX - 0.5;
    for (auto &x : xi) x = rand() / (double)RAND_MAX - 0.5;
    std::vector<float2> regs((size_t)NT * E), smem(SmemSize<N, C>::float2s);
    for (int t = 0; t < NT; ++t)
        for (int e = 0; e < E; ++e) {
            int pt = t / C + e * (N / E), c = t % C;
            regs[(size_t)t * E + e] = make_float2((float)xr[(size_t)pt * C + c], (float)xi[(size_t)pt * C + c]);
        }
    emulate<N, C, E, DIR, 1, R32>(regs, smem, tw.data());
    double err = 0.0, nrm = 0.0;
    for (int c = 0; c < C; ++c)
        for (int t = 0; t < NT; ++t) {
            if (t % C != c) continue;
            for (int e = 0; e < E; ++e) {
                int k = t / C + e * (N / E);
                double sr = 0, si = 0;
                for (int n = 0; n < N; ++n) {
                    double ang = DIR * 2.0 * M_PI * (double)(((long long)k * n) % N) / N;
                    double a = (float)xr[(size_t)n * C + c], b = (float)xi[(size_t)n * C + c];
                    sr += a * cos(ang) - b * sin(ang);
                    si += a * sin(ang) + b * cos(ang);
                }
                float2 g = regs[(size_t)t * E + e];
                err += (g.x - sr) * (g.x - sr) + (g.y - si) * (g.y - si);
                nrm += sr * sr + si * si;
            }
        }
    double rel = sqrt(err / nrm);
    printf("N=%d C=%d E=%d DIR=%d R32=%d rel_l2=%.3e\n", N, C, E, DIR, (int)R32, rel);
    return rel;
}

int main()
{
    double worst = 0.0;
    auto upd = [&](double r) { if (!(r <= worst)) worst = r; };
    upd(check<16, 1, 16, -1>());
    upd(check<32, 2, 16, -1>());
    upd(check<64, 4, 16, +1>());
    upd(check<128, 8, 16, -1>());
    upd(check<256, 1, 16, -1>());
    upd(check<512, 1, 16, +1>());
    upd(check<1024, 4, 16, -1>());
    upd(check<1024, 8, 16, +1>());
    upd(check<2048, 1, 16, -1>());
    upd(check<4096, 1, 16, -1>());
    upd(check<4096, 2, 32, +1>());
    upd(check<1024, 4, 32, -1>());
    upd(check<64, 1, 32, -1>());
    upd(check<8192, 1, 16, +1>());
    upd(check<8192, 1, 32, -1>());
    // the radix-32 first pass of the 8192-point row transforms (32.16.16, padding after every 32 points)
    upd(check<8192, 1, 32, -1, true>());
    upd(check<8192, 1, 32, +1, true>());
    upd(check<32, 1, 32, -1, true>());
    upd(check<512, 1, 32, +1, true>());
    printf("worst=%.3e\n", worst);
    return worst < 2e-6 ? 0 : 1;
}
