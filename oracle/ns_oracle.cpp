// ns_oracle.cpp -- CPU ORACLE for the spectral hyperviscosity Navier-Stokes RHS + SSP-RK3 step.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
// cpu_baseline / --impl reference legs of bench.py may load it.  It shares no code, headers,
// tables or helpers with the CUDA path under paper_2401_09843_b200/csrc/.
//
// It is a plain, slow, step-by-step fp64 restatement of the discretisation in
//   Rohner & Mishra, "Efficient Computation of Large-Scale Statistical Solutions to
//   Incompressible Fluid Flows" (PASC'24, arXiv 2401.09843)  -- cited below as PAPER.md:Lnnn:
//     eq. (2.1)-(2.4)  PAPER.md:L96-116   spectral hyperviscosity discretisation, multiplier Q_N
//     eq. (2.5)        PAPER.md:L122-126  Leray-projected spectral time derivative
//     Algorithm 2      PAPER.md:L128-136  pad -> iFFT -> u(x)u -> FFT -> dealias -> d/dt u_hat
//     eq. (2.6)        PAPER.md:L146-153  third-order SSP Runge-Kutta
// Readings of points where the paper is silent (A1..A20) are listed in DESIGN.md section 3.
//
// Deliberately naive: every 3-D transform is a FULL complex transform on the padded M^3 grid
// (no r2c tricks, no pruning, no fusion), 1-D transforms are a textbook recursive
// decimation-in-time radix-2/3 FFT (O(n^2) DFT for any other prime factor), OpenMP is used only
// over independent 1-D lines / independent wavenumbers.
//
// Parity pins (tests/test_oracle_pins.py): P0 FFT vs O(n^2) DFT and numpy; P1 RHS vs O(N^6) direct
// convolution; P2 Taylor-Green / ABC project to zero; P3 RK3 decay closed form; P4 energy identity;
// P5 div-free; P6 Galilean shift; P7 padding independence; P8 spectrum/Parseval; P9 structure
// function identity; P10 temporal order 3; P11 hyperviscous single mode; P12 orc_rhs_at_modes (direct
// truncated convolution at sampled wavenumbers) vs the step-by-step RHS and vs the test's own O(N^6) sum;
// P13 orc_max_velocity / rhs_parts' umax: constant field (Euclidean norm of all three components), a cosine whose
// maximum lies on the padded grid only, and a zero-padded numpy.fft.irfftn of a random state.
// "parity unpinned" against the authors' code (the paper gives no formula): the readings A3
// (Nyquist planes zero), A5 (form of Q_k), A6 (constants), A10 (CFL formula), A14 (energy-spectrum
// binning), A15 (structure function) -- they are pinned for self-consistency only.

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;
static const double PI = 3.14159265358979323846264338327950288;

// ------------------------------------------------------------------------------------------------
// 1-D transforms.  X[k] = sum_j x[j] exp(sign * 2 pi i j k / n), unnormalised, sign = -1 analysis
// ("forward"), sign = +1 synthesis ("inverse", PAPER.md:L101 writes fields as sum f_k e^{ik.x}).
// ------------------------------------------------------------------------------------------------
// exp(sign * 2 pi i num/den).  The den roots of unity are tabulated once per den (plain cos/sin of
// the reduced argument); the table is only a cache of this formula.
static const cplx* root_table(long den) {
    static std::vector<cplx> tables[4097];
    static bool ready[4097] = {false};
    if (!ready[den]) {
#pragma omp critical(orc_root_table)
        if (!ready[den]) {
            std::vector<cplx> t((size_t)den);
            for (long j = 0; j < den; ++j) {
                const double a = 2.0 * PI * (double)j / (double)den;
                t[(size_t)j] = cplx(std::cos(a), std::sin(a));
            }
            tables[den].swap(t);
#pragma omp flush
            ready[den] = true;
        }
    }
    return tables[den].data();
}
static cplx unit_root(int sign, long num, long den) {
    num %= den;
    if (den > 4096) {
        const double a = 2.0 * PI * (double)num / (double)den;
        return cplx(std::cos(a), sign * std::sin(a));
    }
    const cplx w = root_table(den)[num];
    return sign > 0 ? w : std::conj(w);
}

static void dft_direct(int n, int sign, const cplx* in, long istride, cplx* out, long ostride) {
    for (int k = 0; k < n; ++k) {
        cplx acc(0.0, 0.0);
        for (int j = 0; j < n; ++j) acc += in[j * istride] * unit_root(sign, (long)j * k, n);
        out[k * ostride] = acc;
    }
}

// Recursive decimation in time: n = p*m, p the smallest prime factor in {2,3}:
//   X[k + m*t] = sum_{q<p} w_n^{q(k+mt)} * E_q[k],   E_q = DFT_m(x[q], x[q+p], ...)
static void fft_rec(int n, int sign, const cplx* in, long istride, cplx* out) {
    if (n == 1) { out[0] = in[0]; return; }
    int p = 0;
    if (n % 2 == 0) p = 2; else if (n % 3 == 0) p = 3;
    if (p == 0 || n <= 3) { dft_direct(n, sign, in, istride, out, 1); return; }
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

// In-place 3-D transform of a full complex [n][n][n] array, axis by axis.
static void fft3d(int n, int sign, cplx* a) {
    const long n2 = (long)n * n;
    for (int axis = 0; axis < 3; ++axis) {
        const long stride = axis == 0 ? n2 : (axis == 1 ? n : 1);
#pragma omp parallel
        {
            std::vector<cplx> line((size_t)n), res((size_t)n);
#pragma omp for schedule(static)
            for (long l = 0; l < n2; ++l) {
                const long i = l / n, j = l % n;
                long base;
                if (axis == 0) base = i * n + j;           // (iy, iz) fixed
                else if (axis == 1) base = i * n2 + j;     // (ix, iz) fixed
                else base = i * n2 + j * n;                // (ix, iy) fixed
                for (int t = 0; t < n; ++t) line[t] = a[base + t * stride];
                fft_rec(n, sign, line.data(), 1, res.data());
                for (int t = 0; t < n; ++t) a[base + t * stride] = res[t];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Index conventions (readings A1-A3).  Domain [0,2pi)^3, integer wavenumbers.
// Stored index i on an n-point axis <-> wavenumber k = i (i < n/2), i - n (i > n/2); i == n/2 is
// the Nyquist entry, which is identically zero in state and RHS (A3).
// Half spectrum: [3][N][N][N/2+1] complex, kz = 0..N/2 fastest.
// ------------------------------------------------------------------------------------------------
static inline int wavenumber(int i, int n) { return i < n / 2 ? i : i - n; }
static inline bool nyquist(int i, int n) { return i == n / 2; }
static inline int wrap(int k, int m) { return ((k % m) + m) % m; }

struct Params { double nu, eps, s, m_cut, q_exp; int q_sharp; };

// d_k = nu |k|^2 + eps_N |k|^{2s} Q_k          (eq. 2.1 viscous term; reading A4: damping)
// eps_N = eps / N^{2s-1}                       (eq. 2.4; reading A6)
// Q_k = 0 for |k| <= m_N, else 1 - (m_N/|k|)^q (eq. 2.3 lower bound; reading A5)
// q = (2s-1)/theta, theta = 1/2 by default; m_N = sqrt(N) by default; |k| Euclidean (A7).
static double dissipation(const Params& p, int N, double k2) {
    if (k2 == 0.0) return 0.0;
    double d = p.nu * k2;
    if (p.eps != 0.0) {
        const double kabs = std::sqrt(k2);
        const double mN = p.m_cut < 0.0 ? std::sqrt((double)N) : p.m_cut;
        const double q = p.q_exp < 0.0 ? (2.0 * p.s - 1.0) / 0.5 : p.q_exp;
        double Q = 0.0;
        if (kabs > mN) Q = p.q_sharp ? 1.0 : 1.0 - std::pow(mN / kabs, q);
        const double epsN = p.eps / std::pow((double)N, 2.0 * p.s - 1.0);
        d += epsN * std::pow(kabs, 2.0 * p.s) * Q;
    }
    return d;
}

// Step 2 of Algorithm 2: place the half spectrum of one component into a full
// complex M^3 spectrum at index (k mod M) per axis, Hermitian-completing kz<0 from kz>0; everything
// else zero.  The kz = 0 plane is copied as stored (the physical field is defined as the real part).
static void pad_to_full(int N, int M, const cplx* uh, cplx* full) {
    const int Hs = N / 2 + 1;
    std::fill(full, full + (size_t)M * M * M, cplx(0.0, 0.0));
    for (int ix = 0; ix < N; ++ix) {
        if (nyquist(ix, N)) continue;
        const int kx = wavenumber(ix, N);
        for (int iy = 0; iy < N; ++iy) {
            if (nyquist(iy, N)) continue;
            const int ky = wavenumber(iy, N);
            for (int kz = 0; kz < N / 2; ++kz) {
                const cplx v = uh[((size_t)ix * N + iy) * Hs + kz];
                full[((size_t)wrap(kx, M) * M + wrap(ky, M)) * M + wrap(kz, M)] = v;
                if (kz > 0) full[((size_t)wrap(-kx, M) * M + wrap(-ky, M)) * M + wrap(-kz, M)] = std::conj(v);
            }
        }
    }
}

// Step 3: u_i(X_j) = Re sum_k u_hat_i(k) e^{i k.X_j} on the M^3 grid.
static void to_physical(int N, int M, const cplx* uh_comp, std::vector<cplx>& work, double* u_out) {
    pad_to_full(N, M, uh_comp, work.data());
    fft3d(M, +1, work.data());
    const size_t n = (size_t)M * M * M;
    for (size_t i = 0; i < n; ++i) u_out[i] = work[i].real();
}

// Steps 4-5: B_hat(k) = M^-3 sum_j B(X_j) e^{-i k.X_j}, kept for k in K_N only.
static void to_spectral_truncated(int N, int M, const double* b_phys, std::vector<cplx>& work, cplx* bh) {
    const int Hs = N / 2 + 1;
    const size_t n = (size_t)M * M * M;
    for (size_t i = 0; i < n; ++i) work[i] = cplx(b_phys[i], 0.0);
    fft3d(M, -1, work.data());
    const double scale = 1.0 / ((double)M * M * M);
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < N; ++iy)
            for (int iz = 0; iz < Hs; ++iz) {
                cplx v(0.0, 0.0);
                if (!nyquist(ix, N) && !nyquist(iy, N) && !nyquist(iz, N)) {
                    const int kx = wavenumber(ix, N), ky = wavenumber(iy, N), kz = iz;
                    v = work[((size_t)wrap(kx, M) * M + wrap(ky, M)) * M + wrap(kz, M)] * scale;
                }
                bh[((size_t)ix * N + iy) * Hs + iz] = v;
            }
}

// Whole Algorithm 2 + eq. 2.5.  Outputs (any may be NULL):
//   b_hat  [3][N][N][Hs]  b_i = -i sum_j k_j B_hat_ij
//   n_hat  [3][N][N][Hs]  (1 - k k^T/|k|^2) b                     (eq. 2.5)
//   r_hat  [3][N][N][Hs]  n_hat - d_k u_hat                       (eq. 2.1 viscous term)
//   umax   max over the M^3 grid of |u|_2                         (reading A10)
static void rhs_parts(int N, int M, const Params& p, const cplx* uh, cplx* b_hat, cplx* n_hat, cplx* r_hat,
                      double* umax) {
    const int Hs = N / 2 + 1;
    const size_t ns = (size_t)N * N * Hs, np = (size_t)M * M * M;
    std::vector<cplx> work(np);
    std::vector<double> u(3 * np), B(np);
    for (int c = 0; c < 3; ++c) to_physical(N, M, uh + c * ns, work, u.data() + c * np);
    if (umax) {
        double mx = 0.0;
        for (size_t i = 0; i < np; ++i) {
            const double a = std::sqrt(u[i] * u[i] + u[np + i] * u[np + i] + u[2 * np + i] * u[2 * np + i]);
            if (a > mx) mx = a;
        }
        *umax = mx;
    }
    // Step 3 of Algorithm 2 with the symmetry remark of PAPER.md:L245: six products.
    static const int pi_[6] = {0, 0, 0, 1, 1, 2}, pj_[6] = {0, 1, 2, 1, 2, 2};
    std::vector<cplx> Bh(6 * ns);
    for (int t = 0; t < 6; ++t) {
        const double* a = u.data() + pi_[t] * np;
        const double* b = u.data() + pj_[t] * np;
        for (size_t i = 0; i < np; ++i) B[i] = a[i] * b[i];
        to_spectral_truncated(N, M, B.data(), work, Bh.data() + t * ns);
    }
    static const int sym[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};
#pragma omp parallel for schedule(static)
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < N; ++iy)
            for (int iz = 0; iz < Hs; ++iz) {
                const size_t o = ((size_t)ix * N + iy) * Hs + iz;
                cplx b[3] = {0, 0, 0}, nn[3] = {0, 0, 0}, rr[3] = {0, 0, 0};
                const bool dead = nyquist(ix, N) || nyquist(iy, N) || nyquist(iz, N);
                if (!dead) {
                    const double k[3] = {(double)wavenumber(ix, N), (double)wavenumber(iy, N), (double)iz};
                    const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                    for (int i = 0; i < 3; ++i) {
                        cplx acc(0.0, 0.0);
                        for (int j = 0; j < 3; ++j) acc += k[j] * Bh[sym[i][j] * ns + o];
                        b[i] = cplx(0.0, -1.0) * acc;
                    }
                    if (k2 > 0.0) {  // reading A8: RHS(0) = 0
                        const cplx kb = k[0] * b[0] + k[1] * b[1] + k[2] * b[2];
                        const double d = dissipation(p, N, k2);
                        for (int i = 0; i < 3; ++i) {
                            nn[i] = b[i] - k[i] * kb / k2;
                            rr[i] = nn[i] - d * uh[i * ns + o];
                        }
                    }
                }
                for (int i = 0; i < 3; ++i) {
                    if (b_hat) b_hat[i * ns + o] = b[i];
                    if (n_hat) n_hat[i * ns + o] = nn[i];
                    if (r_hat) r_hat[i * ns + o] = rr[i];
                }
            }
}

extern "C" {

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

// 1-D transforms on interleaved complex arrays (for pin P0).
void orc_dft1d(int n, int sign, const double* in, double* out) {
    dft_direct(n, sign, (const cplx*)in, 1, (cplx*)out, 1);
}
void orc_fft1d(int n, int sign, const double* in, double* out) {
    fft_rec(n, sign, (const cplx*)in, 1, (cplx*)out);
}
// Full complex 3-D transform, in place, [n][n][n] interleaved (for pin P0, 3-D part).
void orc_fft3d(int n, int sign, double* a) { fft3d(n, sign, (cplx*)a); }

double orc_dissipation(int N, double nu, double eps, double s, double m_cut, double q_exp, int q_sharp, double k2) {
    Params p{nu, eps, s, m_cut, q_exp, q_sharp};
    return dissipation(p, N, k2);
}

// RHS and its parts.  u_hat, outputs: [3][N][N][N/2+1] interleaved complex.  M = padded size (3N/2).
void orc_rhs_parts(int N, int M, double nu, double eps, double s, double m_cut, double q_exp, int q_sharp,
                   const double* u_hat, double* b_hat, double* n_hat, double* r_hat, double* umax) {
    Params p{nu, eps, s, m_cut, q_exp, q_sharp};
    rhs_parts(N, M, p, (const cplx*)u_hat, (cplx*)b_hat, (cplx*)n_hat, (cplx*)r_hat, umax);
}

// The plain definition the pseudo-spectral evaluation reaches exactly (up to rounding order): with exact
// dealiasing (reading A3/A12) the truncated transform of the pointwise product is the Galerkin-truncated
// convolution sum  B_hat_ij(k) = sum_{p+q=k; p,q in K_N} u_hat_i(p) u_hat_j(q)  (eq. 2.5, PAPER.md:L124-126:
// F[u (x) u]_k restricted to the retained modes, Algorithm 2 steps 1-5).  Evaluated
// directly, O(N^3) per requested wavenumber, for sampled-output parity at sizes where rhs_parts needs
// too much memory.  modes: [nmodes][3] stored indices (ix, iy, iz), iz <= N/2.  r_out: [nmodes][3] complex.
// The field meant by a half spectrum is the real part of its synthesis, i.e. the kz = 0 plane enters
// through its Hermitian part (same definition as to_physical above).
void orc_rhs_at_modes(int N, double nu, double eps, double s, double m_cut, double q_exp, int q_sharp,
                      const double* u_hat, int nmodes, const int* modes, double* r_out) {
    Params prm{nu, eps, s, m_cut, q_exp, q_sharp};
    const int Hs = N / 2 + 1, K = N / 2 - 1, W = 2 * K + 1;  // wavenumbers -K..K per axis
    const size_t ns = (size_t)N * N * Hs, nf = (size_t)W * W * W;
    const cplx* uh = (const cplx*)u_hat;
    // full spectrum F[c][kx+K][ky+K][kz+K]
    std::vector<cplx> F(3 * nf);
    auto stored = [&](int c, int kx, int ky, int kz) {  // kz >= 0
        return uh[c * ns + ((size_t)wrap(kx, N) * N + wrap(ky, N)) * Hs + kz];
    };
    for (int c = 0; c < 3; ++c)
#pragma omp parallel for schedule(static)
        for (int kx = -K; kx <= K; ++kx)
            for (int ky = -K; ky <= K; ++ky)
                for (int kz = -K; kz <= K; ++kz) {
                    cplx v;
                    if (kz > 0) v = stored(c, kx, ky, kz);
                    else if (kz < 0) v = std::conj(stored(c, -kx, -ky, -kz));
                    else v = 0.5 * (stored(c, kx, ky, 0) + std::conj(stored(c, -kx, -ky, 0)));
                    F[c * nf + ((size_t)(kx + K) * W + (ky + K)) * W + (kz + K)] = v;
                }
    static const int pi_[6] = {0, 0, 0, 1, 1, 2}, pj_[6] = {0, 1, 2, 1, 2, 2};
    static const int sym[3][3] = {{0, 1, 2}, {1, 3, 4}, {2, 4, 5}};
    for (int m = 0; m < nmodes; ++m) {
        const int ix = modes[3 * m], iy = modes[3 * m + 1], iz = modes[3 * m + 2];
        cplx* out = (cplx*)r_out + 3 * m;
        out[0] = out[1] = out[2] = cplx(0.0, 0.0);
        if (nyquist(ix, N) || nyquist(iy, N) || nyquist(iz, N)) continue;
        const int k[3] = {wavenumber(ix, N), wavenumber(iy, N), iz};
        if (k[0] == 0 && k[1] == 0 && k[2] == 0) continue;  // reading A8
        // p ranges over K_N with q = k - p in K_N as well
        const int lo[3] = {std::max(-K, k[0] - K), std::max(-K, k[1] - K), std::max(-K, k[2] - K)};
        const int hi[3] = {std::min(K, k[0] + K), std::min(K, k[1] + K), std::min(K, k[2] + K)};
        long double accr[6] = {0, 0, 0, 0, 0, 0}, acci[6] = {0, 0, 0, 0, 0, 0};
#pragma omp parallel
        {
            long double lr[6] = {0, 0, 0, 0, 0, 0}, li[6] = {0, 0, 0, 0, 0, 0};
#pragma omp for schedule(static) collapse(2)
            for (int px = lo[0]; px <= hi[0]; ++px)
                for (int py = lo[1]; py <= hi[1]; ++py) {
                    cplx row[6] = {0, 0, 0, 0, 0, 0};
                    const size_t op = ((size_t)(px + K) * W + (py + K)) * W + K;
                    const size_t oq = ((size_t)(k[0] - px + K) * W + (k[1] - py + K)) * W + K;
                    for (int pz = lo[2]; pz <= hi[2]; ++pz) {
                        cplx up[3], uq[3];
                        for (int c = 0; c < 3; ++c) {
                            up[c] = F[c * nf + op + pz];
                            uq[c] = F[c * nf + oq + (k[2] - pz)];
                        }
                        for (int t = 0; t < 6; ++t) row[t] += up[pi_[t]] * uq[pj_[t]];
                    }
                    for (int t = 0; t < 6; ++t) { lr[t] += row[t].real(); li[t] += row[t].imag(); }
                }
#pragma omp critical(orc_modes_acc)
            for (int t = 0; t < 6; ++t) { accr[t] += lr[t]; acci[t] += li[t]; }
        }
        cplx Bh[6];
        for (int t = 0; t < 6; ++t) Bh[t] = cplx((double)accr[t], (double)acci[t]);
        const double kd[3] = {(double)k[0], (double)k[1], (double)k[2]};
        const double k2 = kd[0] * kd[0] + kd[1] * kd[1] + kd[2] * kd[2];
        cplx b[3];
        for (int i = 0; i < 3; ++i) {
            cplx acc(0.0, 0.0);
            for (int j = 0; j < 3; ++j) acc += kd[j] * Bh[sym[i][j]];
            b[i] = cplx(0.0, -1.0) * acc;
        }
        const cplx kb = kd[0] * b[0] + kd[1] * b[1] + kd[2] * b[2];
        const double d = dissipation(prm, N, k2);
        for (int i = 0; i < 3; ++i) out[i] = b[i] - kd[i] * kb / k2 - d * stored(i, k[0], k[1], k[2]);
    }
}

// One SSP-RK3 step (eq. 2.6), dissipation explicit inside R (reading A9).
void orc_step(int N, int M, double nu, double eps, double s, double m_cut, double q_exp, int q_sharp,
              double* u_hat, double dt) {
    Params p{nu, eps, s, m_cut, q_exp, q_sharp};
    const size_t n = (size_t)3 * N * N * (N / 2 + 1);
    cplx* u = (cplx*)u_hat;
    std::vector<cplx> R(n), u1(n), u2(n);
    rhs_parts(N, M, p, u, nullptr, nullptr, R.data(), nullptr);
    for (size_t i = 0; i < n; ++i) u1[i] = u[i] + dt * R[i];
    rhs_parts(N, M, p, u1.data(), nullptr, nullptr, R.data(), nullptr);
    for (size_t i = 0; i < n; ++i) u2[i] = 0.75 * u[i] + 0.25 * u1[i] + 0.25 * dt * R[i];
    rhs_parts(N, M, p, u2.data(), nullptr, nullptr, R.data(), nullptr);
    for (size_t i = 0; i < n; ++i) u[i] = (1.0 / 3.0) * u[i] + (2.0 / 3.0) * u2[i] + (2.0 / 3.0) * dt * R[i];
}

// Initialisation (eq. 2.1 third line: u(0) = P_N u_0; reading A11): analysis transform
// of the N^3 samples with 1/N^3, Nyquist planes zeroed, Leray projector applied for k != 0, mean kept.
void orc_set_initial(int N, const double* u_phys, double* u_hat) {
    const int Hs = N / 2 + 1;
    const size_t ns = (size_t)N * N * Hs, np = (size_t)N * N * N;
    cplx* uh = (cplx*)u_hat;
    std::vector<cplx> work(np);
    for (int c = 0; c < 3; ++c) {
        for (size_t i = 0; i < np; ++i) work[i] = cplx(u_phys[c * np + i], 0.0);
        fft3d(N, -1, work.data());
        const double scale = 1.0 / ((double)N * N * N);
        for (int ix = 0; ix < N; ++ix)
            for (int iy = 0; iy < N; ++iy)
                for (int iz = 0; iz < Hs; ++iz) {
                    cplx v = work[((size_t)ix * N + iy) * N + iz] * scale;
                    if (nyquist(ix, N) || nyquist(iy, N) || nyquist(iz, N)) v = cplx(0.0, 0.0);
                    uh[c * ns + ((size_t)ix * N + iy) * Hs + iz] = v;
                }
    }
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < N; ++iy)
            for (int iz = 0; iz < Hs; ++iz) {
                const double k[3] = {(double)wavenumber(ix, N), (double)wavenumber(iy, N), (double)iz};
                const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                if (k2 == 0.0) continue;
                const size_t o = ((size_t)ix * N + iy) * Hs + iz;
                const cplx ku = k[0] * uh[o] + k[1] * uh[ns + o] + k[2] * uh[2 * ns + o];
                for (int i = 0; i < 3; ++i) uh[i * ns + o] -= k[i] * ku / k2;
            }
}

// Physical field on the N grid: u(x_j) = Re sum_k u_hat(k) e^{i k.x_j}; out [3][N][N][N].
void orc_get_fields(int N, const double* u_hat, double* u_phys) {
    const size_t ns = (size_t)N * N * (N / 2 + 1), np = (size_t)N * N * N;
    std::vector<cplx> work(np);
    for (int c = 0; c < 3; ++c) to_physical(N, N, (const cplx*)u_hat + c * ns, work, u_phys + c * np);
}

// max over the padded M^3 grid of the Euclidean |u| (reading A10).
double orc_max_velocity(int N, int M, const double* u_hat) {
    const size_t ns = (size_t)N * N * (N / 2 + 1), np = (size_t)M * M * M;
    std::vector<cplx> work(np);
    std::vector<double> u(3 * np);
    for (int c = 0; c < 3; ++c) to_physical(N, M, (const cplx*)u_hat + c * ns, work, u.data() + c * np);
    double mx = 0.0;
    for (size_t i = 0; i < np; ++i) {
        const double a = std::sqrt(u[i] * u[i] + u[np + i] * u[np + i] + u[2 * np + i] * u[2 * np + i]);
        if (a > mx) mx = a;
    }
    return mx;
}

// Energy spectrum (reading A14): E(K) = 1/2 sum_{K-1/2 <= |k| < K+1/2} |u_hat_k|^2 over the FULL
// spectrum (half-spectrum weight 1 for kz = 0, 2 for kz > 0); modes beyond the last bin are dropped.
void orc_energy_spectrum(int N, const double* u_hat, int nbins, double* E) {
    const int Hs = N / 2 + 1;
    const size_t ns = (size_t)N * N * Hs;
    const cplx* uh = (const cplx*)u_hat;
    for (int b = 0; b < nbins; ++b) E[b] = 0.0;
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < N; ++iy)
            for (int iz = 0; iz < Hs; ++iz) {
                if (nyquist(ix, N) || nyquist(iy, N) || nyquist(iz, N)) continue;
                const double kx = wavenumber(ix, N), ky = wavenumber(iy, N), kz = iz;
                const int bin = (int)std::floor(std::sqrt(kx * kx + ky * ky + kz * kz) + 0.5);
                if (bin >= nbins) continue;
                const size_t o = ((size_t)ix * N + iy) * Hs + iz;
                const double w = iz == 0 ? 1.0 : 2.0;
                E[bin] += 0.5 * w * (std::norm(uh[o]) + std::norm(uh[ns + o]) + std::norm(uh[2 * ns + o]));
            }
}

// Enstrophy spectrum (PAPER.md:L163 names the writer only; reading A20): with the vorticity
// omega_hat_k = i k x u_hat_k,  Z(K) = 1/2 sum_{K-1/2 <= |k| < K+1/2} |omega_hat_k|^2 over the FULL spectrum
// (same shells and weights as orc_energy_spectrum), so that sum_K Z = 1/2 <|curl u|^2>.
void orc_enstrophy_spectrum(int N, const double* u_hat, int nbins, double* Z) {
    const int Hs = N / 2 + 1;
    const size_t ns = (size_t)N * N * Hs;
    const cplx* uh = (const cplx*)u_hat;
    const cplx I(0.0, 1.0);
    for (int b = 0; b < nbins; ++b) Z[b] = 0.0;
    for (int ix = 0; ix < N; ++ix)
        for (int iy = 0; iy < N; ++iy)
            for (int iz = 0; iz < Hs; ++iz) {
                if (nyquist(ix, N) || nyquist(iy, N) || nyquist(iz, N)) continue;
                const double kx = wavenumber(ix, N), ky = wavenumber(iy, N), kz = iz;
                const int bin = (int)std::floor(std::sqrt(kx * kx + ky * ky + kz * kz) + 0.5);
                if (bin >= nbins) continue;
                const size_t o = ((size_t)ix * N + iy) * Hs + iz;
                const cplx u1 = uh[o], u2 = uh[ns + o], u3 = uh[2 * ns + o];
                const cplx w1 = I * (ky * u3 - kz * u2), w2 = I * (kz * u1 - kx * u3), w3 = I * (kx * u2 - ky * u1);
                const double w = iz == 0 ? 1.0 : 2.0;
                Z[bin] += 0.5 * w * (std::norm(w1) + std::norm(w2) + std::norm(w3));
            }
}

// Second-order structure function (reading A15), computed in PHYSICAL space on the N grid:
// S2(l) = (1/3) sum_{d=1..3} < |u(x + l dx e_d) - u(x)|^2 >_x,  l = 1..nl.
void orc_structure_function(int N, const double* u_hat, int nl, double* S2) {
    const size_t np = (size_t)N * N * N;
    std::vector<double> u(3 * np);
    orc_get_fields(N, u_hat, u.data());
    for (int l = 1; l <= nl; ++l) {
        double acc = 0.0;
        for (int ix = 0; ix < N; ++ix)
            for (int iy = 0; iy < N; ++iy)
                for (int iz = 0; iz < N; ++iz) {
                    const size_t o = ((size_t)ix * N + iy) * N + iz;
                    const size_t ox = ((size_t)((ix + l) % N) * N + iy) * N + iz;
                    const size_t oy = ((size_t)ix * N + (iy + l) % N) * N + iz;
                    const size_t oz = ((size_t)ix * N + iy) * N + (iz + l) % N;
                    for (int c = 0; c < 3; ++c) {
                        const double a = u[c * np + o];
                        const double dx = u[c * np + ox] - a, dy = u[c * np + oy] - a, dz = u[c * np + oz] - a;
                        acc += dx * dx + dy * dy + dz * dz;
                    }
                }
        S2[l - 1] = acc / (3.0 * (double)np);
    }
}

// Structure function of order p (PAPER.md:L164 names the writer only; reading A15 extended to p != 2):
// S_p(l) = (1/3) sum_{d=1..3} < |u(x + l dx e_d) - u(x)|^p >_x with the Euclidean norm of the vector increment,
// in PHYSICAL space on the N grid, l = 1..nl.  p = 2 is orc_structure_function.
void orc_structure_function_p(int N, const double* u_hat, double p, int nl, double* Sp) {
    const size_t np = (size_t)N * N * N;
    std::vector<double> u(3 * np);
    orc_get_fields(N, u_hat, u.data());
    for (int l = 1; l <= nl; ++l) {
        double acc = 0.0;
        for (int ix = 0; ix < N; ++ix)
            for (int iy = 0; iy < N; ++iy)
                for (int iz = 0; iz < N; ++iz) {
                    const size_t o = ((size_t)ix * N + iy) * N + iz;
                    const size_t od[3] = {((size_t)((ix + l) % N) * N + iy) * N + iz, ((size_t)ix * N + (iy + l) % N) * N + iz,
                                          ((size_t)ix * N + iy) * N + (iz + l) % N};
                    for (int d = 0; d < 3; ++d) {
                        double r2 = 0.0;
                        for (int c = 0; c < 3; ++c) {
                            const double du = u[c * np + od[d]] - u[c * np + o];
                            r2 += du * du;
                        }
                        acc += std::pow(r2, 0.5 * p);
                    }
                }
        Sp[l - 1] = acc / (3.0 * (double)np);
    }
}

}  // extern "C"
