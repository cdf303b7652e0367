// twiddles_host.h -- host-side construction of the twiddle-table block described in ns_internal.h.
// All roots are evaluated in long double from exactly reduced arguments and rounded once to T.
#pragma once
#include <cmath>
#include <vector>

#include "ns_internal.h"

namespace ns {

// Block layout (complex entries): twA [0,L) twB [L,2L) w3a [2L,3L) w3b [3L,4L) (unused [4L,7L)) z16 [7L,8L) gN [8L,10L).
template <typename T>
inline std::vector<cx<T>> build_twiddle_block(int L) {
    const long double twopi = 6.283185307179586476925286766559005768L;
    int R1 = 0, R2 = 0;
    fft_split(L, &R1, &R2);
    std::vector<cx<T>> h(twiddle_table_len(L));
    for (auto& e : h) { e.x = 0; e.y = 0; }
    auto root = [&](long num, long den) {
        const long double a = twopi * (long double)(num % den) / (long double)den;
        cx<T> w;
        w.x = (T)cosl(a);
        w.y = (T)sinl(a);
        return w;
    };
    for (int r1 = 0; r1 < R1; ++r1)
        for (int n2 = 0; n2 < R2; ++n2) {
            h[(size_t)r1 * R2 + n2] = root((long)r1 * n2, L);
            h[(size_t)L + (size_t)n2 * R1 + r1] = root((long)r1 * n2, L);
        }
    for (int n = 0; n < L; ++n) {
        h[(size_t)2 * L + n] = root(n, 3L * L);
        h[(size_t)3 * L + n] = root(2L * n, 3L * L);
    }
    for (int j = 0; j < 2 * L; ++j) h[(size_t)8 * L + j] = root(j, 2L * L);   // exp(2 pi i j / N), N = 2L
    if (L >= 64 && (L & (L - 1)) == 0) {
        const int G = L / 16;
        for (int r1 = 0; r1 < 16; ++r1)
            for (int t = 0; t < G; ++t) h[(size_t)7 * L + (size_t)r1 * G + t] = root((long)r1 * t, L);
    }
    return h;
}

template <typename T>
inline Twiddles<T> make_twiddles(const cx<T>* base, int L) {
    Twiddles<T> t;
    t.twA = base;
    t.twB = base + L;
    t.w3a = base + 2 * (size_t)L;
    t.w3b = base + 3 * (size_t)L;
    t.z16 = base + 7 * (size_t)L;
    t.gN = base + 8 * (size_t)L;
    return t;
}

}  // namespace ns
