// ns_mg_solver.cu -- host side of the multi-device solver (include/ns_mg.h): one sample distributed over P
// devices by slabs (Algorithm 3), one process driving all of them.  Launch sequences and event ordering
// only; every arithmetic step runs in the kernels of ns.h's path (same launchers, sub-ranges by pointer / stride) and the slab
// exchanges are peer stores of those kernels (ColSplit in kernels_col.cuh).
#include <cmath>
#include <cstdio>
#include <cstring>
#include <initializer_list>
#include <limits>
#include <string>
#include <vector>

#include "../../include/ns_mg.h"
#include "kernels_misc.cuh"
#include "ns_internal.h"
#include "twiddles_host.h"

using namespace ns;

struct ns_mg_solver {
    std::string err;
    long long launches = 0;
    virtual ~ns_mg_solver() {}
    virtual int set_spectral(const void* u) = 0;
    virtual int get_spectral(void* u) = 0;
    virtual int rhs(void* out) = 0;
    virtual int step(bool use_cfl, double dt, double cfl, double t_end, double* dt_out) = 0;
    virtual int max_velocity(double* out) = 0;
    virtual double time() = 0;
    virtual long long exchange_bytes() const = 0;
    virtual long long device_bytes() const = 0;
};

static thread_local std::string g_mg_create_error;

namespace {

// same formula as ns_solver.cu (eq. 2.1 viscous term with the readings A4-A6 of DESIGN.md)
double mg_dissipation_rate(const ns_params& p, int N, double k2) {
    if (k2 <= 0.0) return 0.0;
    double d = p.nu * k2;
    if (p.eps != 0.0) {
        const double kabs = std::sqrt(k2);
        const double mN = p.m_cut < 0.0 ? std::sqrt((double)N) : p.m_cut;
        const double qe = p.q_exp < 0.0 ? (2.0 * p.s - 1.0) * 2.0 : p.q_exp;
        if (kabs > mN) {
            const double Q = p.q_sharp ? 1.0 : 1.0 - std::pow(mN / kabs, qe);
            d += p.eps / std::pow((double)N, 2.0 * p.s - 1.0) * std::pow(k2, p.s) * Q;
        }
    }
    return d;
}

// public [3][N][N][H+1] (whole array on this device) -> the rank's ky slab of the internal layout [3][N][Nyl][H]
template <typename T>
__global__ void mg_to_internal_kernel(const cx<T>* __restrict__ pub, cx<T>* __restrict__ in, int N, int Nyl, int iy0, long total) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int H = N / 2;
    const int iz = (int)(idx % H);
    const int iyl = (int)((idx / H) % Nyl);
    const int ix = (int)((idx / ((long)H * Nyl)) % N);
    const int c = (int)(idx / ((long)H * Nyl * N));
    const int iy = iy0 + iyl;
    cx<T> v = pub[(((long)c * N + ix) * N + iy) * (H + 1) + iz];
    if (ix == N / 2 || iy == N / 2) v = mk<T>(0, 0);
    in[idx] = v;
}
// internal slab [3][N][Nyl][H] -> public slab [3][N][Nyl][H+1] (the kz = N/2 column is zero)
template <typename T>
__global__ void mg_to_public_kernel(const cx<T>* __restrict__ in, cx<T>* __restrict__ pub, int N, int Nyl, long total_pub) {
    const long idx = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total_pub) return;
    const int H = N / 2;
    const int iz = (int)(idx % (H + 1));
    const long row = idx / (H + 1);
    pub[idx] = iz == H ? mk<T>(0, 0) : in[row * H + iz];
}
// time-step bookkeeping of one rank from the max|u|^2 bits of ALL ranks (each rank evaluates the same expression)
static __global__ void mg_dt_kernel(const unsigned long long* um_all, int P, int use_cfl, double dt_given, double cfl, double dx,
                                    double t_end, double* dt, double* t, int* bad) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    unsigned long long m = 0;
    for (int r = 0; r < P; ++r) m = um_all[r] > m ? um_all[r] : m;      // bit order = value order for non-negative doubles
    double v = 0.0;
    if (nonfinite_sq(m)) {
        *bad = 1;
    } else if (!use_cfl) {
        v = dt_given;
    } else {
        const double remaining = t_end - *t;
        if (remaining > 0.0) {
            const double um = sqrt(__longlong_as_double((long long)m));
            v = um > 0.0 ? cfl * dx / um : remaining;
            if (!(v < remaining)) v = remaining;
        }
    }
    *dt = v;
    *t += v;
}

template <typename T>
struct MgRank {
    int dev = 0, num_sms = 0;
    cudaStream_t st = nullptr;
    cx<T>*U = nullptr, *V = nullptr, *X = nullptr, *Tt = nullptr, *Y = nullptr, *Z = nullptr, *B = nullptr, *R = nullptr, *pub = nullptr,
         *twbase = nullptr;
    T* dtab = nullptr;
    double *dt_dev = nullptr, *t_dev = nullptr;
    unsigned long long *umax2 = nullptr, *um_all = nullptr;
    unsigned long long* ptab = nullptr;   // [1 + NS_NFLUX][P] destination base addresses of the fused exchanges (a1; a5 per component)
    int* bad = nullptr;
    cudaEvent_t e1 = nullptr, e2 = nullptr, e5 = nullptr, e6 = nullptr, ez = nullptr;
    std::vector<void*> allocs;
};

template <typename T>
class MgSolver final : public ns_mg_solver {
public:
    int N, L, M, H, P, Nyl, Ml;
    ns_params prm;
    std::vector<MgRank<T>> rk;
    bool has_state = false;
    size_t rank_bytes = 0;

    MgSolver(int N_, int P_, const ns_params& p) : N(N_), L(N_ / 2), M(3 * N_ / 2), H(N_ / 2), P(P_), Nyl(N_ / P_), Ml(3 * N_ / 2 / P_), prm(p), rk((size_t)P_) {}
    ~MgSolver() override {
        for (auto& r : rk) {
            cudaSetDevice(r.dev);
            if (r.st) cudaStreamSynchronize(r.st);
            for (void* p : r.allocs) cudaFree(p);
            cudaEvent_t evs[5] = {r.e1, r.e2, r.e5, r.e6, r.ez};
            for (cudaEvent_t e : evs)
                if (e) cudaEventDestroy(e);
            if (r.st) cudaStreamDestroy(r.st);
        }
    }
    int fail(int code, const std::string& msg) { err = msg; return code; }
    int cuda_fail(cudaError_t e, const char* where) { err = std::string(where) + ": " + cudaGetErrorString(e); return NS_ERR_CUDA; }
#define MG_CK(call)                                           \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)
#define MG_LAUNCH(call, name)                                 \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(e__, name);  \
        ++launches;                                           \
    } while (0)
    static unsigned blocks_for(long total, int threads) { return (unsigned)((total + threads - 1) / threads); }
    Twiddles<T> tw(const MgRank<T>& r) const { return make_twiddles<T>(r.twbase, L); }

    template <typename U> int alloc(MgRank<T>& r, U** p, size_t count) {
        void* q = nullptr;
        cudaError_t e = cudaMalloc(&q, count * sizeof(U));
        if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return fail(NS_ERR_OOM, "device allocation failed"); }
        if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc");
        r.allocs.push_back(q);
        rank_bytes += count * sizeof(U);
        *p = (U*)q;
        return NS_OK;
    }

    int init(const int* devices) {
        int ndev = 0;
        MG_CK(cudaGetDeviceCount(&ndev));
        for (int r = 0; r < P; ++r) {
            if (devices[r] < 0 || devices[r] >= ndev) return fail(NS_ERR_INVALID_ARG, "device ordinal out of range");
            rk[(size_t)r].dev = devices[r];
        }
        // peer access between distinct devices (the slab exchange is direct device-to-device copies)
        for (int r = 0; r < P; ++r)
            for (int s = 0; s < P; ++s) {
                const int a = rk[(size_t)r].dev, b = rk[(size_t)s].dev;
                if (a == b) continue;
                int can = 0;
                MG_CK(cudaDeviceCanAccessPeer(&can, a, b));
                if (!can) return fail(NS_ERR_CUDA, "devices cannot access each other's memory (no peer access)");
                MG_CK(cudaSetDevice(a));
                cudaError_t e = cudaDeviceEnablePeerAccess(b, 0);
                if (e == cudaErrorPeerAccessAlreadyEnabled) cudaGetLastError();
                else if (e != cudaSuccess) return cuda_fail(e, "cudaDeviceEnablePeerAccess");
            }
        const std::vector<cx<T>> htw = build_twiddle_block<T>(L);
        const size_t ndt = (size_t)3 * L * L + 1;
        std::vector<T> hd(ndt);
        for (size_t k2 = 0; k2 < ndt; ++k2) hd[k2] = (T)mg_dissipation_rate(prm, N, (double)k2);
        const size_t sl = (size_t)N * Nyl * H;          // one component of a ky slab
        const size_t pl = (size_t)Ml * N * H;           // one component of a px slab before the y pass
        const size_t pm = (size_t)Ml * M * H;           // ... after it
        for (int r = 0; r < P; ++r) {
            MgRank<T>& k = rk[(size_t)r];
            rank_bytes = 0;
            MG_CK(cudaSetDevice(k.dev));
            MG_CK(cudaDeviceGetAttribute(&k.num_sms, cudaDevAttrMultiProcessorCount, k.dev));
            MG_CK(cudaStreamCreateWithFlags(&k.st, cudaStreamNonBlocking));
            int rc;
            if ((rc = alloc(k, &k.U, 3 * sl)) || (rc = alloc(k, &k.V, 3 * sl)) || (rc = alloc(k, &k.R, 3 * sl)) ||
                (rc = alloc(k, &k.X, NS_NFLUX * (size_t)M * Nyl * H)) || (rc = alloc(k, &k.Tt, 3 * pl)) ||
                (rc = alloc(k, &k.Y, 3 * pm)) || (rc = alloc(k, &k.Z, NS_NFLUX * pm)) || (rc = alloc(k, &k.B, NS_NFLUX * sl)) ||
                (rc = alloc(k, &k.pub, (size_t)3 * N * N * (H + 1))) || (rc = alloc(k, &k.twbase, htw.size())) ||
                (rc = alloc(k, &k.dtab, ndt)) || (rc = alloc(k, &k.dt_dev, 1)) || (rc = alloc(k, &k.t_dev, 1)) ||
                (rc = alloc(k, &k.umax2, 1)) || (rc = alloc(k, &k.um_all, (size_t)P)) || (rc = alloc(k, &k.bad, 1)) ||
                (rc = alloc(k, &k.ptab, (size_t)(1 + NS_NFLUX) * P)))
                return rc;
            MG_CK(cudaMemcpyAsync(k.twbase, htw.data(), htw.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, k.st));
            MG_CK(cudaMemcpyAsync(k.dtab, hd.data(), hd.size() * sizeof(T), cudaMemcpyHostToDevice, k.st));
            MG_CK(cudaMemsetAsync(k.t_dev, 0, sizeof(double), k.st));
            MG_CK(cudaMemsetAsync(k.dt_dev, 0, sizeof(double), k.st));
            MG_CK(cudaMemsetAsync(k.bad, 0, sizeof(int), k.st));
            cudaEvent_t* evs[5] = {&k.e1, &k.e2, &k.e5, &k.e6, &k.ez};
            for (cudaEvent_t* e : evs) MG_CK(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
            MG_CK(cudaStreamSynchronize(k.st));
        }
        // destination tables of the fused exchanges (all ranks' buffers exist now)
        const size_t ncs = (size_t)Nyl * H;
        for (int r = 0; r < P; ++r) {
            MgRank<T>& k = rk[(size_t)r];
            std::vector<unsigned long long> h((size_t)(1 + NS_NFLUX) * P);
            for (int s = 0; s < P; ++s) {
                // a1 of rank r: output row px -> plane px % Ml of Tt_s [3][Ml][N][H], at this rank's ky rows
                h[(size_t)s] = (unsigned long long)(rk[(size_t)s].Tt + (size_t)r * Nyl * H);
                // a5 of rank r, component c: output row ky -> row ky % Nyl of X_s [5][M][Nyl][H], at this rank's px planes
                for (int c = 0; c < NS_NFLUX; ++c)
                    h[(size_t)(1 + c) * P + s] = (unsigned long long)(rk[(size_t)s].X + ((size_t)c * M + (size_t)r * Ml) * ncs);
            }
            MG_CK(cudaSetDevice(k.dev));
            MG_CK(cudaMemcpy(k.ptab, h.data(), h.size() * sizeof(unsigned long long), cudaMemcpyHostToDevice));
        }
        return NS_OK;
    }
    long long device_bytes() const override { return (long long)rank_bytes; }
    long long exchange_bytes() const override {
        // exchange A: 3 components, exchange B: 5; every rank keeps 1/P of its slab, sends (P-1)/P
        return (long long)((3 + NS_NFLUX) * (size_t)M * N * H * sizeof(cx<T>) / P * (P - 1));
    }
    int sync_all() {
        for (auto& k : rk) {
            MG_CK(cudaSetDevice(k.dev));
            MG_CK(cudaStreamSynchronize(k.st));
        }
        return NS_OK;
    }

    // ---------------------------------------------------------------- a1 (+ exchange A) | a2, a3+a4, a5 (+ exchange B) | a6
    // which = 0: transform the state U, 1: the stage state V.  Result: rank r's B = Th [5][N][Nyl][H].
    // Both exchanges are FUSED into the producing pass: a1 of rank r stores output row px straight into Tt of the rank that owns
    // that px plane, a5 of rank s stores output row ky straight into X of the rank that owns that ky row (ColSplit: peer
    // stores over NVLink, overlapped with the butterflies of the next tile); no separate transpose / copy pass exists.
    // Ordering between the rank streams by events: e1 (a1 done), e2 (a2 done: Tt consumed), e5 (a5 done), e6 (a6 done: X consumed).
    int transform(int which, bool want_umax) {
        const long nc = (long)Nyl * H;      // contiguous columns of a ky slab row
        for (int r = 0; r < P; ++r) {
            MgRank<T>& k = rk[(size_t)r];
            MG_CK(cudaSetDevice(k.dev));
            for (int s = 0; s < P; ++s) MG_CK(cudaStreamWaitEvent(k.st, rk[(size_t)s].e2, 0));   // Tt_s of the previous pass consumed
            ColSplit sp;
            sp.rows = Ml;                   // output row px -> rank px / Ml, plane px % Ml of Tt [3][Ml][N][H], at this rank's ky rows
            sp.peer = k.ptab;
            MG_LAUNCH(launch_col_inv<T>(k.st, k.num_sms, L, which ? k.V : k.U, rk[0].Tt + (size_t)r * Nyl * H, nc, 3, nc, (long)N * H, (long)N * nc,
                                        (long)Ml * N * H, tw(k), &sp),
                      "a1 col_inv x + exchange A");
            MG_CK(cudaEventRecord(k.e1, k.st));
        }
        for (int s = 0; s < P; ++s) {       // physical side of rank s
            MgRank<T>& k = rk[(size_t)s];
            MG_CK(cudaSetDevice(k.dev));
            for (int r = 0; r < P; ++r) MG_CK(cudaStreamWaitEvent(k.st, rk[(size_t)r].e1, 0));   // every rank's a1 has stored into Tt_s
            MG_LAUNCH(launch_col_inv<T>(k.st, k.num_sms, L, k.Tt, k.Y, H, (long)3 * Ml, H, H, (long)N * H, (long)M * H, tw(k)), "a2 col_inv y");
            MG_CK(cudaEventRecord(k.e2, k.st));
            MG_LAUNCH(launch_z_fused<T>(k.st, k.num_sms, L, k.Y, k.Z, (long)Ml * M, 1, want_umax ? k.umax2 : nullptr, tw(k)), "a3+a4 z_fused");
            if (want_umax) MG_CK(cudaEventRecord(k.ez, k.st));
            for (int r = 0; r < P; ++r) MG_CK(cudaStreamWaitEvent(k.st, rk[(size_t)r].e6, 0));   // X_r of the previous pass consumed
            for (int c = 0; c < NS_NFLUX; ++c) {
                ColSplit sp;
                sp.rows = Nyl;              // output row ky -> rank ky / Nyl, row ky % Nyl of X [5][M][Nyl][H], at this rank's px planes
                sp.peer = k.ptab + (size_t)(1 + c) * P;
                MG_LAUNCH(launch_col_fwd<T>(k.st, k.num_sms, L, k.Z + (size_t)c * Ml * M * H, rk[0].X + ((size_t)c * M + (size_t)s * Ml) * nc, H,
                                            (long)Ml, H, H, (long)M * H,
                                            nc, (T)1, tw(k), &sp),
                          "a5 col_fwd y + exchange B");
            }
            MG_CK(cudaEventRecord(k.e5, k.st));
        }
        for (int r = 0; r < P; ++r) {       // spectral side of rank r
            MgRank<T>& k = rk[(size_t)r];
            MG_CK(cudaSetDevice(k.dev));
            for (int s = 0; s < P; ++s) MG_CK(cudaStreamWaitEvent(k.st, rk[(size_t)s].e5, 0));   // every rank's a5 has stored into X_r
            MG_LAUNCH(launch_col_fwd<T>(k.st, k.num_sms, L, k.X, k.B, nc, NS_NFLUX, nc, nc, (long)M * nc, (long)N * nc, (T)1, tw(k)),
                      "a6 col_fwd x");
            MG_CK(cudaEventRecord(k.e6, k.st));
        }
        return NS_OK;
    }

    // a7 on every rank's ky slab; sel: 0 = U, 1 = V, 2 = R (output only), -1 = none
    cx<T>* pick(MgRank<T>& k, int sel) { return sel == 0 ? k.U : (sel == 1 ? k.V : (sel == 2 ? k.R : nullptr)); }
    int spectral(int us, int un, int out, double alpha, double beta, double gamma, int mode) {
        const long total = (long)N * Nyl * H;
        const T scale = (T)(1.0 / ((double)M * M * M * z_fused_output_scale(L)));
        for (int r = 0; r < P; ++r) {
            MgRank<T>& k = rk[(size_t)r];
            MG_CK(cudaSetDevice(k.dev));
            spectral_kernel<T><<<blocks_for(total, 256), 256, 0, k.st>>>(k.B, pick(k, us), pick(k, un), pick(k, out), N, N / 2, total, k.dtab, scale,
                                                                          (T)alpha, (T)beta, (T)gamma, k.dt_dev, mode, Nyl, r * Nyl);
            MG_LAUNCH(cudaGetLastError(), "a7 spectral_kernel");
        }
        return NS_OK;
    }

    int step(bool use_cfl, double dt, double cfl, double t_end, double* dt_out) override {
        if (!has_state) return fail(NS_ERR_STATE, "no state set");
        if (use_cfl ? !(cfl > 0.0) : (!(dt == dt) || std::isinf(dt))) return fail(NS_ERR_INVALID_ARG, "need cfl > 0 / a finite dt");
        int rc;
        for (auto& k : rk) {
            MG_CK(cudaSetDevice(k.dev));
            MG_CK(cudaMemsetAsync(k.umax2, 0, sizeof(unsigned long long), k.st));
        }
        if ((rc = transform(0, true)) != NS_OK) return rc;
        for (int r = 0; r < P; ++r) {       // every rank forms the same dt from the maxima of all ranks
            MgRank<T>& k = rk[(size_t)r];
            MG_CK(cudaSetDevice(k.dev));
            for (int s = 0; s < P; ++s) {
                MG_CK(cudaStreamWaitEvent(k.st, rk[(size_t)s].ez, 0));
                MG_CK(cudaMemcpyAsync(k.um_all + s, rk[(size_t)s].umax2, sizeof(unsigned long long), cudaMemcpyDefault, k.st));
            }
            mg_dt_kernel<<<1, 32, 0, k.st>>>(k.um_all, P, use_cfl ? 1 : 0, dt, cfl, 2.0 * 3.14159265358979323846 / N, t_end, k.dt_dev, k.t_dev,
                                             k.bad);
            MG_LAUNCH(cudaGetLastError(), "mg_dt");
        }
        // eq. (2.6)
        if ((rc = spectral(0, -1, 1, 0.0, 1.0, 1.0, 1)) != NS_OK) return rc;
        if ((rc = transform(1, false)) != NS_OK) return rc;
        if ((rc = spectral(1, 0, 1, 0.75, 0.25, 0.25, 1)) != NS_OK) return rc;
        if ((rc = transform(1, false)) != NS_OK) return rc;
        if ((rc = spectral(1, 0, 0, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0, 1)) != NS_OK) return rc;
        if (dt_out) {
            int bad = 0;
            MG_CK(cudaSetDevice(rk[0].dev));
            MG_CK(cudaMemcpyAsync(dt_out, rk[0].dt_dev, sizeof(double), cudaMemcpyDeviceToHost, rk[0].st));
            MG_CK(cudaMemcpyAsync(&bad, rk[0].bad, sizeof(int), cudaMemcpyDeviceToHost, rk[0].st));
            if ((rc = sync_all()) != NS_OK) return rc;
            if (bad) return fail(NS_ERR_NONFINITE, "the velocity field is not finite (NaN or inf); the sample is frozen");
        }
        return NS_OK;
    }

    int max_velocity(double* out) override {
        if (!has_state) return fail(NS_ERR_STATE, "no state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        int rc;
        for (auto& k : rk) {
            MG_CK(cudaSetDevice(k.dev));
            MG_CK(cudaMemsetAsync(k.umax2, 0, sizeof(unsigned long long), k.st));
        }
        if ((rc = transform(0, true)) != NS_OK) return rc;
        if ((rc = sync_all()) != NS_OK) return rc;
        unsigned long long m = 0;
        for (auto& k : rk) {
            unsigned long long v = 0;
            MG_CK(cudaSetDevice(k.dev));
            MG_CK(cudaMemcpy(&v, k.umax2, sizeof v, cudaMemcpyDeviceToHost));
            m = v > m ? v : m;
        }
        double d;
        std::memcpy(&d, &m, sizeof d);
        *out = std::sqrt(d);
        return NS_OK;
    }

    int set_spectral(const void* in) override {
        if (!in) return fail(NS_ERR_INVALID_ARG, "input pointer is NULL");
        const size_t npub = (size_t)3 * N * N * (H + 1);
        const long total = (long)3 * N * Nyl * H;
        for (int r = 0; r < P; ++r) {
            MgRank<T>& k = rk[(size_t)r];
            MG_CK(cudaSetDevice(k.dev));
            MG_CK(cudaMemcpyAsync(k.pub, in, npub * sizeof(cx<T>), cudaMemcpyHostToDevice, k.st));
            mg_to_internal_kernel<T><<<blocks_for(total, 256), 256, 0, k.st>>>(k.pub, k.U, N, Nyl, r * Nyl, total);
            MG_LAUNCH(cudaGetLastError(), "mg_to_internal");
            MG_CK(cudaMemsetAsync(k.bad, 0, sizeof(int), k.st));
        }
        has_state = true;
        return sync_all();
    }
    // every rank converts its slab of `sel` to the public layout and copies it into rows [r Nyl, (r+1) Nyl) of the host array
    int export_slabs(int sel, void* out) {
        const long total_pub = (long)3 * N * Nyl * (H + 1);
        const size_t sz = sizeof(cx<T>);
        for (int r = 0; r < P; ++r) {
            MgRank<T>& k = rk[(size_t)r];
            MG_CK(cudaSetDevice(k.dev));
            mg_to_public_kernel<T><<<blocks_for(total_pub, 256), 256, 0, k.st>>>(pick(k, sel), k.pub, N, Nyl, total_pub);
            MG_LAUNCH(cudaGetLastError(), "mg_to_public");
            MG_CK(cudaMemcpy2DAsync((cx<T>*)out + (size_t)r * Nyl * (H + 1), (size_t)N * (H + 1) * sz, k.pub, (size_t)Nyl * (H + 1) * sz,
                                    (size_t)Nyl * (H + 1) * sz, (size_t)3 * N, cudaMemcpyDeviceToHost, k.st));
        }
        return sync_all();
    }
    int get_spectral(void* out) override {
        if (!has_state) return fail(NS_ERR_STATE, "no state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        return export_slabs(0, out);
    }
    int rhs(void* out) override {
        if (!has_state) return fail(NS_ERR_STATE, "no state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        int rc = transform(0, false);
        if (rc != NS_OK) return rc;
        if ((rc = spectral(0, -1, 2, 0, 0, 0, 0)) != NS_OK) return rc;
        return export_slabs(2, out);
    }
    double time() override {
        double t = std::numeric_limits<double>::quiet_NaN();
        if (cudaSetDevice(rk[0].dev) != cudaSuccess || cudaStreamSynchronize(rk[0].st) != cudaSuccess ||
            cudaMemcpy(&t, rk[0].t_dev, sizeof t, cudaMemcpyDeviceToHost) != cudaSuccess)
            return std::numeric_limits<double>::quiet_NaN();
        return t;
    }
};

template <typename T>
int mg_create_typed(ns_mg_solver** out, int N, int P, const int* devices, const ns_params& p) {
    MgSolver<T>* s = new MgSolver<T>(N, P, p);
    int rc = s->init(devices);
    if (rc == NS_OK) {
        // one pass over the (uninitialised) workspaces: a decomposition the kernels cannot run is rejected here, not at the first step
        for (auto& k : s->rk) {
            cudaSetDevice(k.dev);
            cudaMemsetAsync(k.U, 0, (size_t)3 * N * (N / P) * (N / 2) * sizeof(cx<T>), k.st);
        }
        rc = s->transform(0, false);
        if (rc == NS_OK) rc = s->sync_all();
        if (rc != NS_OK) {
            s->err = "this N / P decomposition is not supported by the pass kernels: " + s->err;
            rc = NS_ERR_INVALID_ARG;
        }
        s->launches = 0;
    }
    if (rc != NS_OK) {
        g_mg_create_error = s->err;
        delete s;
        return rc;
    }
    *out = s;
    return NS_OK;
}

}  // namespace

extern "C" {

int ns_mg_create(ns_mg_solver** out, int N, int P, const int* devices, const ns_params* p, ns_dtype dtype) {
    g_mg_create_error.clear();
    if (!out) { g_mg_create_error = "out is NULL"; return NS_ERR_INVALID_ARG; }
    *out = nullptr;
    if (dtype != NS_F64 && dtype != NS_F32) { g_mg_create_error = "unknown dtype"; return NS_ERR_INVALID_ARG; }
    const int tile = dtype == NS_F32 ? 16 : 8;
    if (!devices || P < 1 || P > 16) { g_mg_create_error = "need 1 <= P <= 16 devices"; return NS_ERR_INVALID_ARG; }
    if (N < 32 || N > 640 || (N % 2) != 0 || !fft_supported(N / 2) || (N / 2) % tile != 0 || N % P != 0 || (3 * N / 2) % P != 0) {
        g_mg_create_error = "N must be a transform grid of ns.h (p 2^a, N/2 a multiple of the column tile) with N and 3N/2 divisible by P";
        return NS_ERR_INVALID_ARG;
    }
    ns_params prm;
    std::memset(&prm, 0, sizeof prm);
    prm.s = 1.0;
    prm.m_cut = -1.0;
    prm.q_exp = -1.0;
    if (p) prm = *p;
    if (!(prm.s >= 1.0) || prm.nu < 0.0 || prm.eps < 0.0 || !(prm.nu == prm.nu) || !(prm.eps == prm.eps)) {
        g_mg_create_error = "params: need s >= 1, nu >= 0, eps >= 0";
        return NS_ERR_INVALID_ARG;
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        g_mg_create_error = std::string("no usable CUDA device (no CPU fallback): ") + (e != cudaSuccess ? cudaGetErrorString(e) : "0 devices");
        return NS_ERR_CUDA;
    }
    int prev = 0;
    cudaGetDevice(&prev);
    const int rc = dtype == NS_F64 ? mg_create_typed<double>(out, N, P, devices, prm) : mg_create_typed<float>(out, N, P, devices, prm);
    cudaSetDevice(prev);
    return rc;
}
int ns_mg_destroy(ns_mg_solver* h) {
    if (!h) return NS_ERR_INVALID_ARG;
    delete h;
    return NS_OK;
}
#define MG_H(h) if (!(h)) return NS_ERR_INVALID_ARG; (h)->err.clear()
int ns_mg_set_spectral(ns_mg_solver* h, const void* u) { MG_H(h); return h->set_spectral(u); }
int ns_mg_get_spectral(ns_mg_solver* h, void* u) { MG_H(h); return h->get_spectral(u); }
int ns_mg_rhs(ns_mg_solver* h, void* out) { MG_H(h); return h->rhs(out); }
int ns_mg_step(ns_mg_solver* h, double dt) { MG_H(h); return h->step(false, dt, 0, 0, nullptr); }
int ns_mg_step_cfl(ns_mg_solver* h, double cfl, double t_end, double* dt_out) { MG_H(h); return h->step(true, 0, cfl, t_end, dt_out); }
int ns_mg_max_velocity(ns_mg_solver* h, double* out) { MG_H(h); return h->max_velocity(out); }
double ns_mg_time(const ns_mg_solver* h) { return h ? const_cast<ns_mg_solver*>(h)->time() : std::numeric_limits<double>::quiet_NaN(); }
long long ns_mg_exchange_bytes(const ns_mg_solver* h) { return h ? h->exchange_bytes() : 0; }
long long ns_mg_kernel_launches(const ns_mg_solver* h) { return h ? h->launches : 0; }
long long ns_mg_device_bytes(const ns_mg_solver* h) { return h ? h->device_bytes() : 0; }
const char* ns_mg_last_error(const ns_mg_solver* h) { return h ? h->err.c_str() : g_mg_create_error.c_str(); }

}  // extern "C"
