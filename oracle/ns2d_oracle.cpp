// ns2d_oracle.cpp -- CPU ORACLE of the TWO-DIMENSIONAL solver.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as ns_oracle.cpp: only tests/, smoke() and bench.py's oracle
// legs may load it; it shares nothing with paper_2401_09843_b200/csrc/).
//
// The paper's solver exists in a two- and a three-dimensional version (section 4: "the 2D solver is validated
// by simulating some analytically known solutions ... the 2D Taylor-Green Vortex, or the vortex patch"; L394, section 7: "both
// two- and three-dimensional large-scale statistical solutions").  This file restates the SAME discretisation on the torus
// [0,2pi)^2, step by step and in the paper's order, with the readings A1..A20 of DESIGN.md section 3 carried over verbatim:
//     eq. (2.1)-(2.4)  PAPER.md:L96-116   spectral hyperviscosity discretisation (d = 2)
//     eq. (2.5)        PAPER.md:L122-126  Leray-projected spectral time derivative
//     Algorithm 2      PAPER.md:L128-136  pad -> iFFT -> u(x)u -> FFT -> dealias -> d/dt u_hat
//     eq. (2.6)        PAPER.md:L146-153  third-order SSP Runge-Kutta
// Layout: spectral [2][N][N/2+1] complex (index [comp][ikx][iky], iky >= 0 fastest: r2c half spectrum along y),
// physical [2][N][N] reals ([comp][ix][iy]).  Normalised coefficients, Nyquist lines zero, |k| Euclidean.
// Deliberately naive: full complex transforms on the padded M^2 grid, all three products u1u1, u1u2, u2u2, its own plain
// recursive radix-2/3 FFT (restated here, nothing is included from ns_oracle.cpp).
//
// Pins (tests/test_oracle2d_pins.py): Q0 transforms vs numpy; Q1 RHS vs O(N^4) direct convolution; Q2 Taylor-Green
// projects to zero and decays at the closed-form RK3 rate; Q3 energy AND enstrophy identities of the dealiased
// nonlinear term; Q4 solenoidal RHS, masks, Galilean shift, padding independence; Q5 the z-independent THREE-dimensional
// oracle run on the same field (the paper's own validation idea); Q6 max|u| (constant field, padded grid,
// zero-padded numpy irfft2); Q7 spectrum / Parseval; Q8 vortex patch: mean flow and circulation conserved.
#include <algorithm>
#include <cmath>
#include <complex>
#include <vector>

typedef std::complex<double> cplx;
namespace {
const double PI = 3.14159265358979323846264338327950288;

cplx unit_root(int sign, long num, long den) {
    num %= den;
    const double a = 2.0 * PI * (double)num / (double)den;
    return cplx(std::cos(a), sign * std::sin(a));
}
// X[k] = sum_j x[j] exp(sign 2 pi i jk/n): recursive decimation in time, radix 2 / 3, O(n^2) otherwise
void fft_rec(int n, int sign, const cplx* in, long istride, cplx* out) {
    if (n == 1) { out[0] = in[0]; return; }
    int p = 0;
    if (n % 2 == 0) p = 2; else if (n % 3 == 0) p = 3;
    if (p == 0 || n <= 3) {
        for (int k = 0; k < n; ++k) {
            cplx acc(0.0, 0.0);
            for (int j = 0; j < n; ++j) acc += in[j * istride] * unit_root(sign, (long)j * k, n);
            out[k] = acc;
        }
        return;
    }
    const int m = n / p;
    std::vector<cplx> sub((size_t)n);
    for (int q = 0; q < p; ++q) fft_rec(m, sign, in + q * istride, istride * p, sub.data() + (size_t)q * m);
    for (int k = 0; k < m; ++k)
        for (int t = 0; t < p; ++t) {
            cplx acc(0.0, 0.0);
            for (int q = 0; q < p; ++q) acc += unit_root(sign, (long)q * (k + (long)m * t), n) * sub[(size_t)q * m + k];
            out[k + m * t] = acc;
        }
}
// in-place 2-D transform of a full complex [n][n] array
void fft2d(int n, int sign, cplx* a) {
    std::vector<cplx> line((size_t)n), res((size_t)n);
    for (int i = 0; i < n; ++i) {                       // along y (contiguous)
        fft_rec(n, sign, a + (size_t)i * n, 1, res.data());
        for (int t = 0; t < n; ++t) a[(size_t)i * n + t] = res[t];
    }
    for (int j = 0; j < n; ++j) {                       // along x
        for (int t = 0; t < n; ++t) line[t] = a[(size_t)t * n + j];
        fft_rec(n, sign, line.data(), 1, res.data());
        for (int t = 0; t < n; ++t) a[(size_t)t * n + j] = res[t];
    }
}
inline int wavenumber(int i, int n) { return i < n / 2 ? i : i - n; }
inline bool nyquist(int i, int n) { return i == n / 2; }
inline int wrap(int k, int m) { return ((k % m) + m) % m; }

struct Params { double nu, eps, s, m_cut, q_exp; int q_sharp; };
// eq. (2.1)-(2.4), readings A4-A7 (same formula as in three dimensions, |k| the Euclidean norm of the 2-D wavenumber)
double dissipation(const Params& p, int N, double k2) {
    if (k2 == 0.0) return 0.0;
    double d = p.nu * k2;
    if (p.eps != 0.0) {
        const double kabs = std::sqrt(k2);
        const double mN = p.m_cut < 0.0 ? std::sqrt((double)N) : p.m_cut;
        const double q = p.q_exp < 0.0 ? (2.0 * p.s - 1.0) / 0.5 : p.q_exp;
        double Q = 0.0;
        if (kabs > mN) Q = p.q_sharp ? 1.0 : 1.0 - std::pow(mN / kabs, q);
        d += p.eps / std::pow((double)N, 2.0 * p.s - 1.0) * std::pow(kabs, 2.0 * p.s) * Q;
    }
    return d;
}
// Algorithm 2 steps 1-2: pad to M^2 (Hermitian completion of ky < 0), synthesis on X_j = 2 pi j / M, real part
void to_physical(int N, int M, const cplx* uh, double* u) {
    const int Hs = N / 2 + 1;
    std::vector<cplx> full((size_t)M * M, cplx(0.0, 0.0));
    for (int ix = 0; ix < N; ++ix) {
        if (nyquist(ix, N)) continue;
        const int kx = wavenumber(ix, N);
        for (int ky = 0; ky < N / 2; ++ky) {
            const cplx v = uh[(size_t)ix * Hs + ky];
            full[(size_t)wrap(kx, M) * M + wrap(ky, M)] = v;
            if (ky > 0) full[(size_t)wrap(-kx, M) * M + wrap(-ky, M)] = std::conj(v);
        }
    }
    fft2d(M, +1, full.data());
    for (size_t i = 0; i < (size_t)M * M; ++i) u[i] = full[i].real();
}
// steps 4-5: analysis with 1/M^2, kept for k in K_N only
void to_spectral_truncated(int N, int M, const double* b, cplx* bh) {
    const int Hs = N / 2 + 1;
    std::vector<cplx> work((size_t)M * M);
    for (size_t i = 0; i < (size_t)M * M; ++i) work[i] = cplx(b[i], 0.0);
    fft2d(M, -1, work.data());
    const double scale = 1.0 / ((double)M * M);
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < Hs; ++iy) {
            cplx v(0.0, 0.0);
            if (!nyquist(ix, N) && !nyquist(iy, N)) v = work[(size_t)wrap(wavenumber(ix, N), M) * M + iy] * scale;
            bh[(size_t)ix * Hs + iy] = v;
        }
}
// Algorithm 2 + eq. 2.5 + viscous term; any output may be NULL
void rhs_parts(int N, int M, const Params& p, const cplx* uh, cplx* b_hat, cplx* n_hat, cplx* r_hat, double* umax) {
    const int Hs = N / 2 + 1;
    const size_t ns = (size_t)N * Hs, np = (size_t)M * M;
    std::vector<double> u(2 * np), B(np);
    for (int c = 0; c < 2; ++c) to_physical(N, M, uh + c * ns, u.data() + c * np);
    if (umax) {
        double mx = 0.0;
        for (size_t i = 0; i < np; ++i) mx = std::max(mx, std::sqrt(u[i] * u[i] + u[np + i] * u[np + i]));
        *umax = mx;
    }
    static const int pi_[3] = {0, 0, 1}, pj_[3] = {0, 1, 1};       // B11, B12, B22 (upper triangle)
    std::vector<cplx> Bh(3 * ns);
    for (int t = 0; t < 3; ++t) {
        for (size_t i = 0; i < np; ++i) B[i] = u[pi_[t] * np + i] * u[pj_[t] * np + i];
        to_spectral_truncated(N, M, B.data(), Bh.data() + t * ns);
    }
    static const int sym[2][2] = {{0, 1}, {1, 2}};
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < Hs; ++iy) {
            const size_t o = (size_t)ix * Hs + iy;
            cplx b[2] = {0, 0}, nn[2] = {0, 0}, rr[2] = {0, 0};
            if (!nyquist(ix, N) && !nyquist(iy, N)) {
                const double k[2] = {(double)wavenumber(ix, N), (double)iy};
                const double k2 = k[0] * k[0] + k[1] * k[1];
                for (int i = 0; i < 2; ++i) b[i] = cplx(0.0, -1.0) * (k[0] * Bh[sym[i][0] * ns + o] + k[1] * Bh[sym[i][1] * ns + o]);
                if (k2 > 0.0) {
                    const cplx kb = k[0] * b[0] + k[1] * b[1];
                    const double d = dissipation(p, N, k2);
                    for (int i = 0; i < 2; ++i) {
                        nn[i] = b[i] - k[i] * kb / k2;
                        rr[i] = nn[i] - d * uh[i * ns + o];
                    }
                }
            }
            for (int i = 0; i < 2; ++i) {
                if (b_hat) b_hat[i * ns + o] = b[i];
                if (n_hat) n_hat[i * ns + o] = nn[i];
                if (r_hat) r_hat[i * ns + o] = rr[i];
            }
        }
}
}  // namespace

extern "C" {

void orc2_fft2d(int n, int sign, double* a) { fft2d(n, sign, (cplx*)a); }

void orc2_rhs_parts(int N, int M, double nu, double eps, double s, double m_cut, double q_exp, int q_sharp, const double* u_hat,
                    double* b_hat, double* n_hat, double* r_hat, double* umax) {
    Params p{nu, eps, s, m_cut, q_exp, q_sharp};
    rhs_parts(N, M, p, (const cplx*)u_hat, (cplx*)b_hat, (cplx*)n_hat, (cplx*)r_hat, umax);
}

// One SSP-RK3 step (eq. 2.6), dissipation explicit inside R (reading A9)
void orc2_step(int N, int M, double nu, double eps, double s, double m_cut, double q_exp, int q_sharp, double* u_hat, double dt) {
    Params p{nu, eps, s, m_cut, q_exp, q_sharp};
    const size_t n = (size_t)2 * N * (N / 2 + 1);
    cplx* u = (cplx*)u_hat;
    std::vector<cplx> R(n), u1(n), u2(n);
    rhs_parts(N, M, p, u, nullptr, nullptr, R.data(), nullptr);
    for (size_t i = 0; i < n; ++i) u1[i] = u[i] + dt * R[i];
    rhs_parts(N, M, p, u1.data(), nullptr, nullptr, R.data(), nullptr);
    for (size_t i = 0; i < n; ++i) u2[i] = 0.75 * u[i] + 0.25 * u1[i] + 0.25 * dt * R[i];
    rhs_parts(N, M, p, u2.data(), nullptr, nullptr, R.data(), nullptr);
    for (size_t i = 0; i < n; ++i) u[i] = (1.0 / 3.0) * u[i] + (2.0 / 3.0) * u2[i] + (2.0 / 3.0) * dt * R[i];
}

// u(0) = P_N u_0 (eq. 2.1 third line; reading A11): analysis with 1/N^2, Nyquist lines zeroed, Leray projector for k != 0
void orc2_set_initial(int N, const double* u_phys, double* u_hat) {
    const int Hs = N / 2 + 1;
    const size_t ns = (size_t)N * Hs, np = (size_t)N * N;
    cplx* uh = (cplx*)u_hat;
    std::vector<cplx> work(np);
    for (int c = 0; c < 2; ++c) {
        for (size_t i = 0; i < np; ++i) work[i] = cplx(u_phys[c * np + i], 0.0);
        fft2d(N, -1, work.data());
        for (int ix = 0; ix < N; ++ix)
            for (int iy = 0; iy < Hs; ++iy) {
                cplx v = work[(size_t)ix * N + iy] / ((double)N * N);
                if (nyquist(ix, N) || nyquist(iy, N)) v = cplx(0.0, 0.0);
                uh[c * ns + (size_t)ix * Hs + iy] = v;
            }
    }
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < Hs; ++iy) {
            const double k[2] = {(double)wavenumber(ix, N), (double)iy};
            const double k2 = k[0] * k[0] + k[1] * k[1];
            if (k2 == 0.0) continue;
            const size_t o = (size_t)ix * Hs + iy;
            const cplx ku = k[0] * uh[o] + k[1] * uh[ns + o];
            for (int i = 0; i < 2; ++i) uh[i * ns + o] -= k[i] * ku / k2;
        }
}

void orc2_get_fields(int N, const double* u_hat, double* u_phys) {
    const size_t ns = (size_t)N * (N / 2 + 1), np = (size_t)N * N;
    for (int c = 0; c < 2; ++c) to_physical(N, N, (const cplx*)u_hat + c * ns, u_phys + c * np);
}

// max over the padded M^2 grid of the Euclidean |u| (reading A10)
double orc2_max_velocity(int N, int M, const double* u_hat) {
    const size_t ns = (size_t)N * (N / 2 + 1), np = (size_t)M * M;
    std::vector<double> u(2 * np);
    for (int c = 0; c < 2; ++c) to_physical(N, M, (const cplx*)u_hat + c * ns, u.data() + c * np);
    double mx = 0.0;
    for (size_t i = 0; i < np; ++i) mx = std::max(mx, std::sqrt(u[i] * u[i] + u[np + i] * u[np + i]));
    return mx;
}

// Ring spectra (reading A14 in two dimensions): E(K) = 1/2 sum_{K-1/2 <= |k| < K+1/2} |u_hat_k|^2 over the FULL spectrum
// (weight 1 for ky = 0, 2 for ky > 0); enstrophy: |u_hat|^2 replaced by |omega_hat|^2, omega_hat = i (kx u2 - ky u1).
void orc2_spectrum(int N, const double* u_hat, int nbins, int enstrophy, double* E) {
    const int Hs = N / 2 + 1;
    const size_t ns = (size_t)N * Hs;
    const cplx* uh = (const cplx*)u_hat;
    for (int b = 0; b < nbins; ++b) E[b] = 0.0;
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < Hs; ++iy) {
            if (nyquist(ix, N) || nyquist(iy, N)) continue;
            const double kx = wavenumber(ix, N), ky = iy;
            const int bin = (int)std::floor(std::sqrt(kx * kx + ky * ky) + 0.5);
            if (bin >= nbins) continue;
            const size_t o = (size_t)ix * Hs + iy;
            const double e = enstrophy ? std::norm(kx * uh[ns + o] - ky * uh[o]) : std::norm(uh[o]) + std::norm(uh[ns + o]);
            E[bin] += 0.5 * (iy == 0 ? 1.0 : 2.0) * e;
        }
}

}  // extern "C"
