// Host-side pieces of the GPUQT library that need no GPU: input validation, the sliced-ELL
// builder and the Bessel coefficient table (a9).  Product code; shares nothing
// with oracle/.
#pragma once
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/gpuqt.h"

namespace gpuqt {

inline double host_min_image(double d, double box) {
    if (box > 0.0) {
        if (d > 0.5 * box) d -= box;
        else if (d < -0.5 * box) d += box;
    }
    return d;
}

// Validation of the paper's four data sets.  Returns a gpuqt_status and a message.
// n_halo > 0: the table is a row slab of a decomposed lattice -- columns may point at the halo rows
// N .. N + n_halo - 1 (values owned by another slab; x has N + n_halo entries), and Hermiticity can only be
// checked for the entries whose column is an owned row.
inline int validate_inputs(int64_t N, int32_t K, const int32_t* cnt, const int32_t* idx,
                           const double* hre, const double* him, const double* onsite,
                           const double* x, double box, double dE, std::string& msg, int64_t n_halo = 0) {
    if (N <= 0 || K <= 0 || !cnt || !idx || !x || !(dE > 0.0) || n_halo < 0 || N + n_halo > 0x7fffffffLL) {
        msg = "invalid argument (N, K_max, energy_scale must be positive; nbr_count, nbr_index, x required; N < 2^31)";
        return GPUQT_ERR_ARG;
    }
    if (him && !hre) {
        msg = "hop_im given without hop_re";
        return GPUQT_ERR_ARG;
    }
    // index range [A11]
    for (int64_t m = 0; m < N; ++m) {
        const int32_t c = cnt[m];
        if (c < 0 || c > K) {
            msg = "neighbour count out of range at site " + std::to_string(m);
            return GPUQT_ERR_INDEX;
        }
        for (int32_t k = 0; k < c; ++k) {
            const int32_t n = idx[(size_t)m * K + k];
            if (n < 0 || n >= N + n_halo) {
                msg = "neighbour index out of range at site " + std::to_string(m);
                return GPUQT_ERR_INDEX;
            }
        }
    }
    auto H = [&](int64_t m, int32_t k, double& re, double& im) {
        re = hre ? hre[(size_t)m * K + k] : -1.0;
        im = him ? him[(size_t)m * K + k] : 0.0;
    };
    // Hermiticity, bit-exact [A10]: the number of entries (m -> n, h) in row m equals the number
    // of entries (n -> m, conj h) in row n.  Gershgorin bound [A9].  Ambiguous image [A6].
    for (int64_t m = 0; m < N; ++m) {
        double g = onsite ? std::fabs(onsite[m]) : 0.0;
        for (int32_t k = 0; k < cnt[m]; ++k) {
            const int32_t n = idx[(size_t)m * K + k];
            double re, im;
            H(m, k, re, im);
            g += std::hypot(re, im);
            if (re == 0.0 && im == 0.0) continue;
            int here = 0, there = 0;
            for (int32_t j = 0; j < cnt[m]; ++j) {
                double r2, i2;
                H(m, j, r2, i2);
                if (idx[(size_t)m * K + j] == n && r2 == re && i2 == im) ++here;
            }
            for (int32_t j = 0; n < N && j < cnt[n]; ++j) {
                double r2, i2;
                H(n, j, r2, i2);
                if (idx[(size_t)n * K + j] == (int32_t)m && r2 == re && i2 == -im) ++there;
            }
            if (n < N && here != there) {
                msg = "H is not Hermitian: entry (" + std::to_string(m) + "," + std::to_string(n) + ") has no conjugate partner";
                return GPUQT_ERR_NOT_HERMITIAN;
            }
            if (box > 0.0 && std::fabs(x[n] - x[m]) == 0.5 * box) {
                msg = "ambiguous minimum image: |X_n - X_m| == box_length/2 for hop (" + std::to_string(m) + "," + std::to_string(n) + ")";
                return GPUQT_ERR_POSITION;
            }
        }
        if (g > dE) {
            msg = "Gershgorin bound " + std::to_string(g) + " at site " + std::to_string(m) + " exceeds energy_scale " + std::to_string(dE);
            return GPUQT_ERR_SCALE;
        }
    }
    return GPUQT_OK;
}

// Packed sliced-ELL table on the host (layout: kernels.cuh).  A slice is 32 rows; its record is
//   double hre[w][32] (nd >= 1) | double him[w][32] (nd == 2) | double onsite[32] | int32 col[w][32]
// with w the largest neighbour count in the slice and nd the doubles stored per entry: 2 complex,
// 1 real, 0 when every listed hopping is the same real number (hop_const; the paper's default
// "all hoppings -1", and every clean-lattice model) -- then padding is col = N, the
// all-zero row every device vector carries.  If padding every record to K_max costs less
// than 1/16 extra bytes the table is stored uniform (w = K_max everywhere), which lets the
// kernels compute record offsets arithmetically and unroll the neighbour walk.  The record array is
// padded with all-padding records to a multiple of `pad_to` slices, so that a tile of several
// consecutive slices is always one contiguous copy.
struct SellHost {
    int64_t n_slices = 0;               // real slices, ceil(N / 32)
    int uniform = 1;                    // every record has width K_max
    int nd = 1;                         // doubles per entry: 0 constant hopping, 1 real, 2 complex
    double hop_const = 0.0;
    int idx16 = 0;                      // constant hopping with 16-bit columns (see try_idx16): 1 plain, 2 with 0xffff padding entries
    int64_t n_slices_padded = 0;        // records stored: n_slices rounded up to a multiple of pad_to (all-padding records behind)
    std::vector<long long> slice_off;   // [n_slices_padded + 1] byte offsets of the records
    std::vector<unsigned char> rec;
};

inline long long host_record_bytes(int w, int nd) { return 32LL * (8LL * w * nd + 8 + 4LL * w); }

// Re-encode a uniform constant-hopping table (records: onsite[32] | int32 col[K][32]) with 16-bit
// columns: record = double onsite[32] | int32 base[8] | uint16 delta[K][32], col = base[k] + delta, and
// delta = 0xffff stands for a padding entry (col = N, the zero row).  Possible when K <= 8 and, inside
// every (slice, k), the real columns spread less than 65535.  Returns false and leaves the table
// untouched otherwise.
struct SellHost;
inline bool try_idx16(SellHost& s, int K, int64_t N);

// true (and the value) if hop_im is absent and all listed hoppings carry the same bit pattern
inline bool constant_hopping(int64_t N, int32_t K, const int32_t* cnt, const double* hre, const double* him,
                             double& value) {
    if (him) return false;
    if (!hre) {
        value = -1.0;
        return true;
    }
    bool have = false;
    for (int64_t m = 0; m < N; ++m)
        for (int32_t k = 0; k < cnt[m]; ++k) {
            const double h = hre[(size_t)m * K + k];
            if (!have) {
                value = h;
                have = true;
            } else if (std::memcmp(&h, &value, sizeof(double)) != 0) {
                return false;
            }
        }
    if (!have) value = 0.0;
    return true;
}

// pad_col = index of the all-zero vector row (N; N + n_halo for a row slab)
inline void build_sell(int64_t N, int32_t K, const int32_t* cnt, const int32_t* idx,
                       const double* hre, const double* him, const double* onsite, bool allow_const,
                       int pad_to, SellHost& s, int64_t pad_col = -1) {
    if (pad_col < 0) pad_col = N;
    s.nd = him ? 2 : 1;
    if (allow_const && constant_hopping(N, K, cnt, hre, him, s.hop_const)) s.nd = 0;
    const int cplx = s.nd;   // doubles per entry
    s.n_slices = (N + 31) / 32;
    s.n_slices_padded = (s.n_slices + pad_to - 1) / pad_to * pad_to;
    std::vector<int> width((size_t)s.n_slices_padded, 0);
    long long ragged = 0;
    for (int64_t sl = 0; sl < s.n_slices; ++sl) {
        int w = 0;
        for (int64_t m = sl * 32; m < std::min<int64_t>(N, sl * 32 + 32); ++m) w = std::max(w, cnt[m]);
        width[(size_t)sl] = w;
        ragged += host_record_bytes(w, cplx);
    }
    const long long padded = (long long)s.n_slices * host_record_bytes(K, cplx);
    s.uniform = (padded <= ragged + ragged / 16) ? 1 : 0;
    s.slice_off.assign((size_t)s.n_slices_padded + 1, 0);
    for (int64_t sl = 0; sl < s.n_slices_padded; ++sl) {
        if (s.uniform) width[(size_t)sl] = K;
        s.slice_off[(size_t)sl + 1] = s.slice_off[(size_t)sl] + host_record_bytes(width[(size_t)sl], cplx);
    }
    s.rec.assign((size_t)s.slice_off[(size_t)s.n_slices_padded], 0);
    for (int64_t sl = 0; sl < s.n_slices_padded; ++sl) {
        const int w = width[(size_t)sl];
        unsigned char* base = s.rec.data() + s.slice_off[(size_t)sl];
        double* r_hre = reinterpret_cast<double*>(base);
        double* r_him = r_hre + (size_t)w * 32;
        double* r_on = r_hre + (size_t)w * 32 * s.nd;
        int32_t* r_col = reinterpret_cast<int32_t*>(r_on + 32);
        for (int lane = 0; lane < 32; ++lane) {
            const int64_t m = sl * 32 + lane;
            r_on[lane] = (m < N && onsite) ? onsite[m] : 0.0;
            for (int k = 0; k < w; ++k) {
                const size_t e = (size_t)k * 32 + lane;
                if (m < N && k < cnt[m]) {
                    r_col[e] = idx[(size_t)m * K + k];
                    if (s.nd >= 1) r_hre[e] = hre ? hre[(size_t)m * K + k] : -1.0;
                    if (s.nd == 2) r_him[e] = him[(size_t)m * K + k];
                } else if (s.nd == 0) {
                    r_col[e] = (int32_t)pad_col;                               // padding: the zero row
                } else {
                    r_col[e] = (int32_t)(m < N ? m : N - 1);                   // padding: own row, hop 0
                }
            }
        }
    }
}

// J_m(x), m < n, by Miller's backward recurrence normalised with J_0 + 2 sum_k J_2k = 1.
// (Deliberately a different routine from the oracle's libm jn().)
inline void bessel_j_table(double x, int n, std::vector<double>& J) {
    J.assign((size_t)n, 0.0);
    if (n <= 0) return;
    x = std::fabs(x);
    if (x == 0.0) {
        J[0] = 1.0;
        return;
    }
    const int top = std::max(n, (int)std::ceil(x));
    int M = top + 40 + (int)std::ceil(4.0 * std::sqrt((double)top));
    M += (M & 1);   // even
    std::vector<long double> f((size_t)M + 2, 0.0L);
    f[(size_t)M] = 1e-300L;
    const long double xl = (long double)x;
    for (int k = M; k >= 1; --k) {
        f[(size_t)k - 1] = (2.0L * k / xl) * f[(size_t)k] - f[(size_t)k + 1];
        if (fabsl(f[(size_t)k - 1]) > 1e+3000L) {
            for (int j = k - 1; j <= M; ++j) f[(size_t)j] *= 1e-3000L;
        }
    }
    long double norm = f[0];
    for (int k = 2; k <= M; k += 2) norm += 2.0L * f[(size_t)k];
    for (int k = 0; k < n; ++k) J[(size_t)k] = (double)(f[(size_t)k] / norm);
}

// c_m = (2 - delta_0m) (-i sgn dt)^m J_m(dE |dt|)   PAPER.md:154 Eq. 17, :162 Eq. 20 [A8]
inline void bessel_coeffs(double dE, double dt, int order, std::vector<double>& cr, std::vector<double>& ci) {
    std::vector<double> J;
    bessel_j_table(dE * std::fabs(dt), order, J);
    cr.assign((size_t)order, 0.0);
    ci.assign((size_t)order, 0.0);
    const double sg = dt < 0 ? -1.0 : 1.0;
    for (int m = 0; m < order; ++m) {
        const double j = (m == 0 ? 1.0 : 2.0) * J[(size_t)m];
        switch (m & 3) {
        case 0: cr[(size_t)m] = j; break;
        case 1: ci[(size_t)m] = -sg * j; break;
        case 2: cr[(size_t)m] = -j; break;
        default: ci[(size_t)m] = sg * j; break;
        }
    }
}

}  // namespace gpuqt

namespace gpuqt {
inline bool try_idx16(SellHost& s, int K, int64_t N) {
    if (s.nd != 0 || !s.uniform || K > 8) return false;
    const size_t old_bytes = 256 + 128 * (size_t)K, new_bytes = 288 + 64 * (size_t)K;
    std::vector<unsigned char> out((size_t)s.n_slices_padded * new_bytes, 0);
    bool any_pad = false;
    for (int64_t sl = 0; sl < s.n_slices_padded; ++sl) {
        const unsigned char* src = s.rec.data() + (size_t)sl * old_bytes;
        unsigned char* dst = out.data() + (size_t)sl * new_bytes;
        std::memcpy(dst, src, 256);                                            // onsite
        const int32_t* col = reinterpret_cast<const int32_t*>(src + 256);
        int32_t* base = reinterpret_cast<int32_t*>(dst + 256);
        uint16_t* delta = reinterpret_cast<uint16_t*>(dst + 288);
        for (int k = 0; k < K; ++k) {
            int64_t lo = N, hi = -1;                                           // over the real columns (padding is col = N)
            for (int lane = 0; lane < 32; ++lane) {
                const int32_t c = col[k * 32 + lane];
                if (c >= N) continue;
                lo = std::min<int64_t>(lo, c);
                hi = std::max<int64_t>(hi, c);
            }
            if (hi < 0) lo = N;                                                // nothing but padding: base = N, delta = 0
            if (hi - lo > 65534) return false;                                 // 0xffff is reserved for the zero row
            base[k] = (int32_t)lo;
            for (int lane = 0; lane < 32; ++lane) {
                const int32_t c = col[k * 32 + lane];
                // a padding entry is an ordinary delta when the zero row is in reach, else the sentinel
                const bool sentinel = c >= N && (int64_t)N - lo > 65534;
                delta[k * 32 + lane] = sentinel ? (uint16_t)0xffffu : (uint16_t)(c - lo);
                any_pad = any_pad || sentinel;
            }
        }
    }
    s.rec.swap(out);
    for (int64_t sl = 0; sl <= s.n_slices_padded; ++sl) s.slice_off[(size_t)sl] = (long long)((size_t)sl * new_bytes);
    s.idx16 = any_pad ? 2 : 1;
    return true;
}
}  // namespace gpuqt

namespace gpuqt {
// Implicit stencil (kHopStencil in kernels.cuh): re-encode a uniform constant-hopping table
// (records: onsite[32] | int32 col[K][32]) as  record = onsite[32],  pid[slice],  dict[pattern][K][32]  with
// dict = the distinct arrays  rel[k][lane] = col - 32 slice  of the table.  On a regular lattice in natural
// order the relative columns repeat from slice to slice and differ only where a periodic wrap falls into
// the slice, so a few hundred patterns describe millions of rows; vacancies, open edges in the bulk or a
// shuffled numbering make every slice its own pattern and the table is left as it is (returns false).
//   force = false: only when the dictionary is at most 1/16 of the index array it replaces (and <= 8 MB,
//                  so that it stays L2 resident);  force = true: whenever the table is uniform (tests).
struct StencilHost {
    std::vector<int32_t> pid;           // [n_slices_padded]
    std::vector<int32_t> dict;          // [n_patterns][K][32]
    int64_t n_patterns = 0;
};
inline bool try_stencil(SellHost& s, int K, int64_t N, bool force, StencilHost& st) {
    (void)N;
    if (s.nd != 0 || !s.uniform || s.idx16) return false;
    const size_t old_bytes = 256 + 128 * (size_t)K, pat = (size_t)K * 32;
    const size_t index_bytes = (size_t)s.n_slices_padded * pat * 4;
    size_t max_patterns = (size_t)s.n_slices_padded;
    if (!force) max_patterns = std::min<size_t>(index_bytes / 16, (size_t)8 << 20) / (pat * 4);
    std::unordered_map<std::string, int32_t> seen;
    std::vector<int32_t> rel(pat);
    st.pid.assign((size_t)s.n_slices_padded, 0);
    st.dict.clear();
    for (int64_t sl = 0; sl < s.n_slices_padded; ++sl) {
        const int32_t* col = reinterpret_cast<const int32_t*>(s.rec.data() + (size_t)sl * old_bytes + 256);
        for (size_t e = 0; e < pat; ++e) rel[e] = (int32_t)((int64_t)col[e] - sl * 32);
        std::string key(reinterpret_cast<const char*>(rel.data()), pat * 4);
        auto it = seen.find(key);
        if (it == seen.end()) {
            if (seen.size() >= max_patterns) return false;
            it = seen.emplace(std::move(key), (int32_t)seen.size()).first;
            st.dict.insert(st.dict.end(), rel.begin(), rel.end());
        }
        st.pid[(size_t)sl] = it->second;
    }
    st.n_patterns = (int64_t)seen.size();
    std::vector<unsigned char> out((size_t)s.n_slices_padded * 256);
    for (int64_t sl = 0; sl < s.n_slices_padded; ++sl)
        std::memcpy(out.data() + (size_t)sl * 256, s.rec.data() + (size_t)sl * old_bytes, 256);      // onsite
    s.rec.swap(out);
    for (int64_t sl = 0; sl <= s.n_slices_padded; ++sl) s.slice_off[(size_t)sl] = (long long)sl * 256;
    return true;
}
}  // namespace gpuqt

namespace gpuqt {
// Site reordering for locality (round 2): a simple-cubic periodic lattice in natural order (i = x + Lx (y + Ly z), every
// row with its 6 nearest neighbours in any order -- the Anderson model of PAPER.md:353-355 in three dimensions) has
// only the +-x neighbours of a row inside the row's 32-row slice; stored in bricks of 4 x 4 x 2 sites per slice, 4 of
// the 6 neighbours of an average row are in its own slice (shared memory) and the gather stream from L2 halves
// (c4: KPM step 156.7 -> 148.4 us, evolve_msd 456.8 -> 437.0 us).  Square lattices gain nothing from 2-D bricks
// (measured: c2 11.65 vs 11.68 us, the paper's example 5.1 50.2 vs 49.9 us), so only d = 3 is recognised.
// Returns true and the two permutations when the table is such a lattice with Lx, Ly multiples of 4 and Lz even.
inline bool detect_cubic_bricks(int64_t N, int32_t K, const int32_t* cnt, const int32_t* idx,
                                std::vector<int32_t>& new_of_old, std::vector<int32_t>& old_of_new) {
    if (K != 6 || N < 27 || N > 0x7fffffffLL) return false;
    if (cnt[0] != 6) return false;
    int64_t a[6];
    for (int k = 0; k < 6; ++k) a[k] = idx[k];
    std::sort(a, a + 6);
    // neighbours of site 0: 1, Lx - 1, Lx, Lx (Ly - 1), Lx Ly, N - Lx Ly
    const int64_t Lx = a[2];
    if (a[0] != 1 || Lx < 3 || a[1] != Lx - 1 || a[3] % Lx != 0) return false;
    const int64_t Ly = a[3] / Lx + 1, LxLy = Lx * Ly;
    if (Ly < 3 || a[4] != LxLy || N % LxLy != 0) return false;
    const int64_t Lz = N / LxLy;
    if (Lz < 3 || a[5] != N - LxLy) return false;
    if (Lx % 4 || Ly % 4 || Lz % 2) return false;
    for (int64_t m = 0; m < N; ++m) {                 // every row: exactly the six periodic neighbours, in any order
        if (cnt[m] != 6) return false;
        const int64_t x = m % Lx, y = (m / Lx) % Ly, z = m / LxLy;
        int64_t want[6] = {m - x + (x + 1) % Lx, m - x + (x + Lx - 1) % Lx,
                           m - y * Lx + ((y + 1) % Ly) * Lx, m - y * Lx + ((y + Ly - 1) % Ly) * Lx,
                           m - z * LxLy + ((z + 1) % Lz) * LxLy, m - z * LxLy + ((z + Lz - 1) % Lz) * LxLy};
        int64_t have[6];
        for (int k = 0; k < 6; ++k) have[k] = idx[(size_t)m * 6 + k];
        std::sort(want, want + 6);
        std::sort(have, have + 6);
        for (int k = 0; k < 6; ++k)
            if (want[k] != have[k]) return false;
    }
    new_of_old.resize((size_t)N);
    old_of_new.resize((size_t)N);
    const int64_t nbx = Lx / 4, nby = Ly / 4;
    for (int64_t m = 0; m < N; ++m) {
        const int64_t x = m % Lx, y = (m / Lx) % Ly, z = m / LxLy;
        const int64_t brick = (x / 4) + nbx * ((y / 4) + nby * (z / 2));
        const int64_t local = (x % 4) + 4 * ((y % 4) + 4 * (z % 2));
        const int64_t p = brick * 32 + local;
        new_of_old[(size_t)m] = (int32_t)p;
        old_of_new[(size_t)p] = (int32_t)m;
    }
    return true;
}
}  // namespace gpuqt

