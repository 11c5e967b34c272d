// =====================================================================================
// fmm_oracle.cpp  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, fp64 CPU restatement of the adaptive point-charge Laplace FMM of
// arXiv 2511.15269 (jaxFMM), written from /root/reference/PAPER.md only.  It shares no
// code, header, table or constant generator with the CUDA path under
// paper_2511_15269_b200/csrc and is imported only by tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs.
//
// Every function cites the PAPER.md passage it follows.  Where the paper is silent,
// garbled or ambiguous the reading of DESIGN.md ("Readings", T1-T7, L1-L5, E1-E7,
// G1-G5, S1-S7) is used and named.  Nothing is blocked, fused or reordered beyond what
// those passages state; OpenMP loops run over independent target boxes only, so the
// arithmetic order inside every result is the same for any thread count.
//
// Parity pins (tests/test_oracle_*.py): regular/singular basis vs associated-Legendre
// closed forms; grad vs finite differences; addition theorem; Wigner-d vs d^1, d(0),
// orthogonality; rotations vs recomputation from rotated points; M2M/L2L exactness;
// M2L convergence; tree brute force + PAPER.md:50 counts; list partition identity and
// the theta=0.7637 cube pin; whole FMM vs O(N^2) direct sum.
// Cross-level (level-marching) lists: partition identity over all level pairs, symmetry of
// the covered particle pairs, accuracy vs the O(N^2) sum and the count reduction against same-level lists.
// Adjoint evaluate: dot-product identity against the forward evaluate to round-off, the plain definition
// with sources and targets exchanged, symmetry of the single-set same-level operator (tests/test_oracle_adjoint.py).
// "parity unpinned": the interaction counts of Table I -- the helix point set is not given.
//
// Build: g++ -O2 -std=c++17 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/build.py)
// Coefficient layout: K=(p+1)^2 doubles, index(n,m) = n*n + n + m, -n<=m<=n;
// m>=0 <-> real part, m<0 <-> imaginary part.
// =====================================================================================
#include <algorithm>
#include <cfloat>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

inline int IDX(int n, int m) { return n * n + n + m; }
inline int sgn(int m) { return m >= 0 ? 1 : -1; }  // sgn(0)=+1
inline int iabs(int m) { return m < 0 ? -m : m; }

double factorial(int n) {
    double f = 1.0;
    for (int i = 2; i <= n; ++i) f *= (double)i;
    return f;
}

// integer power, 0^0 = 1
double ipow(double b, int e) {
    double r = 1.0;
    for (int i = 0; i < e; ++i) r *= b;
    return r;
}

// -------------------------------------------------------------------------------------
// App. A.1: real regular basis R^_n^m by recursion.
// -------------------------------------------------------------------------------------
void regular_basis(int p, double x, double y, double z, double* R) {
    const double r2 = x * x + y * y + z * z;
    R[IDX(0, 0)] = 1.0;
    if (p >= 1) {
        R[IDX(1, 1)] = x / 2.0;
        R[IDX(1, -1)] = -y / 2.0;
    }
    for (int n = 2; n <= p; ++n) {
        R[IDX(n, n)] = (x * R[IDX(n - 1, n - 1)] + y * R[IDX(n - 1, 1 - n)]) / (2.0 * n);
        R[IDX(n, -n)] = (x * R[IDX(n - 1, 1 - n)] - y * R[IDX(n - 1, n - 1)]) / (2.0 * n);
    }
    for (int n = 0; n <= p - 1; ++n) {
        R[IDX(n + 1, n)] = z * R[IDX(n, n)];
        R[IDX(n + 1, -n)] = z * R[IDX(n, -n)];
    }
    for (int n = 2; n <= p; ++n)
        for (int m = 2 - n; m <= n - 2; ++m)
            R[IDX(n, m)] = ((2.0 * n - 1.0) * z * R[IDX(n - 1, m)] - r2 * R[IDX(n - 2, m)]) /
                           (double)((n - iabs(m)) * (n + iabs(m)));
}

// -------------------------------------------------------------------------------------
// App. A.2: real singular basis S^_n^m by recursion.
// -------------------------------------------------------------------------------------
void singular_basis(int p, double x, double y, double z, double* S) {
    const double r2 = x * x + y * y + z * z;
    const double r = std::sqrt(r2);
    S[IDX(0, 0)] = 1.0 / r;
    if (p >= 1) {
        S[IDX(1, 1)] = x / (r2 * r);
        S[IDX(1, -1)] = y / (r2 * r);
    }
    for (int n = 2; n <= p; ++n) {
        S[IDX(n, n)] = (2.0 * n - 1.0) * (x * S[IDX(n - 1, n - 1)] - y * S[IDX(n - 1, 1 - n)]) / r2;
        S[IDX(n, -n)] = (2.0 * n - 1.0) * (x * S[IDX(n - 1, 1 - n)] + y * S[IDX(n - 1, n - 1)]) / r2;
    }
    for (int n = 0; n <= p - 1; ++n) {
        S[IDX(n + 1, n)] = (2.0 * n + 1.0) * z * S[IDX(n, n)] / r2;
        S[IDX(n + 1, -n)] = (2.0 * n + 1.0) * z * S[IDX(n, -n)] / r2;
    }
    for (int n = 2; n <= p; ++n)
        for (int m = 2 - n; m <= n - 2; ++m)
            S[IDX(n, m)] = ((2.0 * n - 1.0) * z * S[IDX(n - 1, m)] -
                            (double)((n - 1 - m) * (n - 1 + m)) * S[IDX(n - 2, m)]) / r2;
}

// -------------------------------------------------------------------------------------
// App. A.3: gradient of the regular basis; G[3*idx + {0,1,2}].
// Reading G1: PAPER.md:419 is printed with a leading minus; it is the derivative of
// PAPER.md:368 and therefore carries NO minus (pinned by finite differences).
// R must hold regular_basis(p, x, y, z).
// -------------------------------------------------------------------------------------
void regular_grad(int p, double x, double y, double z, const double* R, double* G) {
    const double r2 = x * x + y * y + z * z;
    const double rv[3] = {x, y, z};
    for (int c = 0; c < 3; ++c) G[3 * IDX(0, 0) + c] = 0.0;
    if (p >= 1) {
        for (int c = 0; c < 3; ++c) { G[3 * IDX(1, 1) + c] = 0.0; G[3 * IDX(1, -1) + c] = 0.0; }
        G[3 * IDX(1, 1) + 0] = 0.5;
        G[3 * IDX(1, -1) + 1] = -0.5;
    }
    for (int n = 2; n <= p; ++n) {  // PAPER.md:419-421 (G1)
        for (int c = 0; c < 3; ++c) {
            const double ex = (c == 0) ? 1.0 : 0.0, ey = (c == 1) ? 1.0 : 0.0;
            G[3 * IDX(n, n) + c] = (x * G[3 * IDX(n - 1, n - 1) + c] + y * G[3 * IDX(n - 1, 1 - n) + c] +
                                    R[IDX(n - 1, n - 1)] * ex + R[IDX(n - 1, 1 - n)] * ey) / (2.0 * n);
            G[3 * IDX(n, -n) + c] = (x * G[3 * IDX(n - 1, 1 - n) + c] - y * G[3 * IDX(n - 1, n - 1) + c] +
                                     R[IDX(n - 1, 1 - n)] * ex - R[IDX(n - 1, n - 1)] * ey) / (2.0 * n);
        }
    }
    for (int n = 0; n <= p - 1; ++n) {
        for (int c = 0; c < 3; ++c) {
            const double ez = (c == 2) ? 1.0 : 0.0;
            G[3 * IDX(n + 1, n) + c] = z * G[3 * IDX(n, n) + c] + R[IDX(n, n)] * ez;
            G[3 * IDX(n + 1, -n) + c] = z * G[3 * IDX(n, -n) + c] + R[IDX(n, -n)] * ez;
        }
    }
    for (int n = 2; n <= p; ++n)
        for (int m = 2 - n; m <= n - 2; ++m)
            for (int c = 0; c < 3; ++c) {
                const double ez = (c == 2) ? 1.0 : 0.0;
                G[3 * IDX(n, m) + c] = ((2.0 * n - 1.0) * (z * G[3 * IDX(n - 1, m) + c] + R[IDX(n - 1, m)] * ez) -
                                        r2 * G[3 * IDX(n - 2, m) + c] - 2.0 * R[IDX(n - 2, m)] * rv[c]) /
                                       (double)(n * n - m * m);
            }
}

// -------------------------------------------------------------------------------------
// Wigner small-d, d^j_{m',m}(beta).  The paper delegates to [14];
// reading S6: the textbook explicit sum
//   d^j_{m'm} = sum_s (-1)^{m'-m+s} sqrt((j+m)!(j-m)!(j+m')!(j-m')!) /
//               ((j+m-s)! s! (m'-m+s)! (j-m'-s)!) cos(b/2)^{2j+m-m'-2s} sin(b/2)^{m'-m+2s}
// over all s with non-negative factorial arguments.
// -------------------------------------------------------------------------------------
double wigner_d(int j, int mp, int m, double beta) {
    const double cb = std::cos(0.5 * beta), sb = std::sin(0.5 * beta);
    const double pref = std::sqrt(factorial(j + m) * factorial(j - m) * factorial(j + mp) * factorial(j - mp));
    const int smin = std::max(0, m - mp), smax = std::min(j + m, j - mp);
    double sum = 0.0;
    for (int s = smin; s <= smax; ++s) {
        const double den = factorial(j + m - s) * factorial(s) * factorial(mp - m + s) * factorial(j - mp - s);
        const double sign = ((mp - m + s) % 2 == 0) ? 1.0 : -1.0;
        sum += sign * pref / den * ipow(cb, 2 * j + m - mp - 2 * s) * ipow(sb, mp - m + 2 * s);
    }
    return sum;
}

// -------------------------------------------------------------------------------------
// App. B.1: azimuthal rotation by dphi, for all m including negative
// (E-rules: C' = C cos(m dphi) - C^{-m} sin(m dphi);  D' = D cos + D^{-m} sin).
// -------------------------------------------------------------------------------------
void rot_azimuthal(int p, int local_type, const double* in, double dphi, double* out) {
    for (int n = 0; n <= p; ++n)
        for (int m = -n; m <= n; ++m) {
            const double c = std::cos(m * dphi), s = std::sin(m * dphi);
            out[IDX(n, m)] = local_type ? in[IDX(n, m)] * c + in[IDX(n, -m)] * s
                                        : in[IDX(n, m)] * c - in[IDX(n, -m)] * s;
        }
}

// -------------------------------------------------------------------------------------
// App. B.2: polar rotation by dtheta.  Reading G2: the cases of W are
// "k>0", "k=0 and m>=0", "k=0 and m<0 -> 0"; d_{n,k}^{|m|} = d^n_{m'=|m|, m=k}.
//   C'_n^m = sum_{k=0}^n C_n^{sgn(m)k} N W,   D'_n^m = sum_k D_n^{sgn(m)k} W / N,
//   N = sqrt((n-k)!(n+k)! / ((n-|m|)!(n+|m|)!)).
// -------------------------------------------------------------------------------------
void rot_polar(int p, int local_type, const double* in, double dtheta, double* out) {
    for (int n = 0; n <= p; ++n)
        for (int m = -n; m <= n; ++m) {
            const int am = iabs(m);
            double acc = 0.0;
            for (int k = 0; k <= n; ++k) {
                double W;
                if (k > 0) W = wigner_d(n, am, k, dtheta) + sgn(m) * ((k % 2 == 0) ? 1.0 : -1.0) * wigner_d(n, am, -k, dtheta);
                else if (m >= 0) W = wigner_d(n, am, 0, dtheta);
                else continue;  // k=0, m<0: term absent
                const double N = std::sqrt(factorial(n - k) * factorial(n + k) / (factorial(n - am) * factorial(n + am)));
                const double v = in[IDX(n, sgn(m) * k)];
                acc += local_type ? v * W / N : v * N * W;
            }
            out[IDX(n, m)] = acc;
        }
}

// -------------------------------------------------------------------------------------
// App. B.3: shifts along +z by r > 0 (reading G3: b = old centre -
// new centre, brought onto +z by the preceding rotations).
// -------------------------------------------------------------------------------------
void shift_m2m(int p, const double* C, double r, double* out) {
    for (int n = 0; n <= p; ++n)
        for (int m = -n; m <= n; ++m) {
            double acc = 0.0;
            for (int k = iabs(m); k <= n; ++k) acc += ipow(r, n - k) / factorial(n - k) * C[IDX(k, m)];
            out[IDX(n, m)] = acc;
        }
}
void shift_m2l(int p, const double* C, double r, double* out) {
    for (int n = 0; n <= p; ++n)
        for (int m = -n; m <= n; ++m) {
            double acc = 0.0;
            for (int k = iabs(m); k <= p; ++k) {
                const double sign = (((k + m) % 2 + 2) % 2 == 0) ? 1.0 : -1.0;
                acc += sgn(m) * sign * factorial(n + k) / ipow(r, n + k + 1) * C[IDX(k, m)];
            }
            out[IDX(n, m)] = acc;
        }
}
void shift_l2l(int p, const double* D, double r, double* out) {
    for (int n = 0; n <= p; ++n)
        for (int m = -n; m <= n; ++m) {
            double acc = 0.0;
            for (int k = n; k <= p; ++k) acc += ipow(-r, k - n) / factorial(k - n) * D[IDX(k, m)];
            out[IDX(n, m)] = acc;
        }
}

// -------------------------------------------------------------------------------------
// PAPER.md:154 "rotate -> transform -> rotate back" (rule T_X of DESIGN.md).
// b = old expansion centre - new expansion centre (G3).  (r,theta,phi) of b; forward:
// azimuthal by phi, polar by theta (b now on +z); z-shift of length r; inverse: polar
// by -theta, azimuthal by -phi.  kind: 0=M2M, 1=M2L, 2=L2L.  phi:=0 when b_x=b_y=0 (S7).
// -------------------------------------------------------------------------------------
void translate(int kind, int p, const double* in, const double b[3], double* out) {
    const int K = (p + 1) * (p + 1);
    const double r = std::sqrt(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]);
    std::vector<double> t1(K), t2(K);
    if (r == 0.0) {  // degenerate (single-child chains with identical bbox): identity for M2M/L2L
        std::memcpy(out, in, sizeof(double) * K);
        return;
    }
    double ct = b[2] / r;
    if (ct > 1.0) ct = 1.0;
    if (ct < -1.0) ct = -1.0;
    const double theta = std::acos(ct);
    const double phi = (b[0] == 0.0 && b[1] == 0.0) ? 0.0 : std::atan2(b[1], b[0]);
    const int in_local = (kind == 2) ? 1 : 0;
    const int out_local = (kind == 0) ? 0 : 1;
    rot_azimuthal(p, in_local, in, phi, t1.data());
    rot_polar(p, in_local, t1.data(), theta, t2.data());
    if (kind == 0) shift_m2m(p, t2.data(), r, t1.data());
    else if (kind == 1) shift_m2l(p, t2.data(), r, t1.data());
    else shift_l2l(p, t2.data(), r, t1.data());
    rot_polar(p, out_local, t1.data(), -theta, t2.data());
    rot_azimuthal(p, out_local, t2.data(), -phi, out);
}

// -------------------------------------------------------------------------------------
// Hierarchy, PAPER.md:40-43 and Listing 2; rules T1-T7 of DESIGN.md.
// -------------------------------------------------------------------------------------
int tree_depth(int64_t N, int N_max, int s) {  // T1: smallest l with ceil(N/2^{sl}) <= N_max
    for (int L = 0;; ++L) {
        int64_t q = N;  // ceil(ceil(a/2)/2) = ceil(a/4): repeated ceiling-halving is ceil(N/2^{sL})
        for (int i = 0; i < s * L; ++i) q = (q + 1) / 2;
        if (q <= N_max) return L;
    }
}

struct Tree {
    int64_t N = 0;
    int s = 0, L = 0;
    std::vector<int64_t> perm;                       // tree order -> original index (T4)
    std::vector<int64_t> level_off;                  // global id offset of each level (L+2 entries)
    std::vector<int64_t> box_start, box_count;       // per global box id, range in tree order
    std::vector<double> lo, hi, ctr, rad;            // per global box: 3,3,3,1 (T6); empty boxes: NaN-free zeros, count 0
};

void split_rec(const double* pos, std::vector<int64_t>& ids, int d, int dmax, const std::vector<int64_t>& nd,
               std::vector<std::vector<int64_t>>& leaves) {
    if (d == dmax) {
        std::sort(ids.begin(), ids.end());  // T4 / PAPER.md:220
        leaves.push_back(ids);
        return;
    }
    const int64_t c = (int64_t)ids.size();
    int axis = 0;
    if (c > 0) {  // T3: tight bbox, extent in fp64, longest axis, ties -> lowest axis index
        double e[3];
        for (int a = 0; a < 3; ++a) {
            double mn = pos[3 * ids[0] + a], mx = mn;
            for (int64_t i : ids) { mn = std::min(mn, pos[3 * i + a]); mx = std::max(mx, pos[3 * i + a]); }
            e[a] = mx - mn;
        }
        if (e[1] > e[axis]) axis = 1;
        if (e[2] > e[axis]) axis = 2;
    }
    // order by (coordinate on axis, original index)  (S4)
    std::sort(ids.begin(), ids.end(), [&](int64_t a, int64_t b) {
        const double xa = pos[3 * a + axis], xb = pos[3 * b + axis];
        if (xa < xb) return true;
        if (xb < xa) return false;
        return a < b;
    });
    // upper child gets the last floor(n_d/2), lower child the rest (T3; Listing 2)
    int64_t n_up = nd[d] / 2;
    if (n_up > c) n_up = c;
    std::vector<int64_t> lower(ids.begin(), ids.end() - n_up), upper(ids.end() - n_up, ids.end());
    split_rec(pos, lower, d + 1, dmax, nd, leaves);
    split_rec(pos, upper, d + 1, dmax, nd, leaves);
}

void build_tree(const double* pos, int64_t N, int N_max, int s, Tree& T) {
    T.N = N; T.s = s; T.L = tree_depth(N, N_max, s);
    const int dmax = s * T.L;
    std::vector<int64_t> nd(dmax + 1);
    nd[0] = N;
    for (int d = 0; d < dmax; ++d) nd[d + 1] = (nd[d] + 1) / 2;  // padded row length of Listing 2
    std::vector<int64_t> ids(N);
    for (int64_t i = 0; i < N; ++i) ids[i] = i;
    std::vector<std::vector<int64_t>> leaves;
    split_rec(pos, ids, 0, dmax, nd, leaves);
    T.perm.clear();
    const int64_t n_leaves = (int64_t)1 << dmax;
    std::vector<int64_t> leaf_start(n_leaves + 1, 0);
    for (int64_t b = 0; b < n_leaves; ++b) {
        for (int64_t i : leaves[b]) T.perm.push_back(i);
        leaf_start[b + 1] = (int64_t)T.perm.size();
    }
    T.level_off.assign(T.L + 2, 0);
    for (int l = 0; l <= T.L; ++l) T.level_off[l + 1] = T.level_off[l] + ((int64_t)1 << (s * l));
    const int64_t nb = T.level_off[T.L + 1];
    T.box_start.assign(nb, 0); T.box_count.assign(nb, 0);
    T.lo.assign(3 * nb, 0.0); T.hi.assign(3 * nb, 0.0); T.ctr.assign(3 * nb, 0.0); T.rad.assign(nb, 0.0);
    for (int l = 0; l <= T.L; ++l) {
        const int64_t nbl = (int64_t)1 << (s * l);
        const int64_t leaves_per_box = n_leaves / nbl;  // T2: box b at level l = leaves [b*lpb, (b+1)*lpb)
        for (int64_t b = 0; b < nbl; ++b) {
            const int64_t g = T.level_off[l] + b;
            const int64_t st = leaf_start[b * leaves_per_box], en = leaf_start[(b + 1) * leaves_per_box];
            T.box_start[g] = st; T.box_count[g] = en - st;
            if (en == st) continue;  // T5
            for (int a = 0; a < 3; ++a) {
                double mn = pos[3 * T.perm[st] + a], mx = mn;
                for (int64_t k = st; k < en; ++k) { mn = std::min(mn, pos[3 * T.perm[k] + a]); mx = std::max(mx, pos[3 * T.perm[k] + a]); }
                T.lo[3 * g + a] = mn; T.hi[3 * g + a] = mx;
                T.ctr[3 * g + a] = 0.5 * (mn + mx);  // T6/T7
            }
            const double dx = T.hi[3 * g] - T.lo[3 * g], dy = T.hi[3 * g + 1] - T.lo[3 * g + 1], dz = T.hi[3 * g + 2] - T.lo[3 * g + 2];
            T.rad[g] = 0.5 * std::sqrt((dx * dx + dy * dy) + dz * dz);  // T6, summed x->y->z
        }
    }
}

// eq. (4), rule L1: R + theta r < theta d, strict.
bool admissible(const Tree& T, int64_t ga, int64_t gb, double theta) {
    const double ra = T.rad[ga], rb = T.rad[gb];
    const double R = std::max(ra, rb), r = std::min(ra, rb);
    const double dx = T.ctr[3 * ga] - T.ctr[3 * gb], dy = T.ctr[3 * ga + 1] - T.ctr[3 * gb + 1], dz = T.ctr[3 * ga + 2] - T.ctr[3 * gb + 2];
    const double d = std::sqrt((dx * dx + dy * dy) + dz * dz);
    return R + theta * r < theta * d;
}

struct Lists {
    // CSR by target global box id (L4); sources are global ids, ascending within a row.
    std::vector<int64_t> weak_off; std::vector<int64_t> weak_src;
    // CSR by target leaf (index within leaf level); sources are leaf indices, ascending.
    std::vector<int64_t> strong_off; std::vector<int64_t> strong_src;
};

// PAPER.md:72-74, rules L2-L5 (cross_level = 0), and the level-marching generalisation PAPER.md:82-89 (cross_level = 1,
// reading S9 of DESIGN.md): candidate pairs (target box on level lt, source box on level ls) start at (root, root) with
// lt = ls = 0; admissible candidates (eq. (4)) become weak pairs of their target; the others are refined and re-tested.
//   cross_level = 0: both boxes are refined together, (lt, ls) = (0,0), (1,1), ..., (L,L).
//   cross_level = 1: one side at a time.  "Increase the level with the larger average box radius; if equal, increase the
//     source level; if there are no more source levels, increase the target level".  Sources and targets
//     share one hierarchy here, whose mean box radius shrinks from level to level, so the rule yields the fixed sequence
//     (lt, ls) = (0,0), (0,1), (1,1), (1,2), ..., (L-1,L), (L,L): refine the sources, then the targets, alternately.
// Pairs still failing at (L,L) are the strong leaf pairs (L3).
void build_lists(const Tree& T, double theta, Lists& Ls, int cross_level = 0) {
    const int s = T.s, L = T.L;
    const int64_t nch = (int64_t)1 << s;
    const int64_t nb = T.level_off[L + 1];
    std::vector<std::vector<int64_t>> weak_rows(nb);
    const int64_t n_leaves = (int64_t)1 << (s * L);
    std::vector<std::vector<int64_t>> strong_rows(n_leaves);
    std::vector<std::pair<int64_t, int64_t>> cand, fail;
    cand.push_back({0, 0});  // (root, root), level-local indices (target, source)
    int lt = 0, ls = 0;
    for (;;) {
        fail.clear();
        for (auto& pr : cand) {
            const int64_t ga = T.level_off[lt] + pr.first, gb = T.level_off[ls] + pr.second;
            if (admissible(T, ga, gb, theta)) weak_rows[ga].push_back(gb);
            else fail.push_back(pr);
        }
        if (lt == L && ls == L) break;
        const bool refine_src = cross_level ? (ls == lt) : true;
        const bool refine_tgt = cross_level ? (ls != lt) : true;
        cand.clear();
        for (auto& pr : fail)
            for (int64_t i = 0; i < (refine_tgt ? nch : 1); ++i)
                for (int64_t j = 0; j < (refine_src ? nch : 1); ++j) {
                    const int64_t a = refine_tgt ? pr.first * nch + i : pr.first, b = refine_src ? pr.second * nch + j : pr.second;
                    if (T.box_count[T.level_off[lt + (refine_tgt ? 1 : 0)] + a] == 0 || T.box_count[T.level_off[ls + (refine_src ? 1 : 0)] + b] == 0)
                        continue;  // T5
                    cand.push_back({a, b});
                }
        if (refine_tgt) ++lt;
        if (refine_src) ++ls;
    }
    for (auto& pr : fail) strong_rows[pr.first].push_back(pr.second);  // L3, includes (t,t)
    Ls.weak_off.assign(nb + 1, 0); Ls.weak_src.clear();
    for (int64_t g = 0; g < nb; ++g) {
        std::sort(weak_rows[g].begin(), weak_rows[g].end());
        for (int64_t v : weak_rows[g]) Ls.weak_src.push_back(v);
        Ls.weak_off[g + 1] = (int64_t)Ls.weak_src.size();
    }
    Ls.strong_off.assign(n_leaves + 1, 0); Ls.strong_src.clear();
    for (int64_t t = 0; t < n_leaves; ++t) {
        std::sort(strong_rows[t].begin(), strong_rows[t].end());
        for (int64_t v : strong_rows[t]) Ls.strong_src.push_back(v);
        Ls.strong_off[t + 1] = (int64_t)Ls.strong_src.size();
    }
}

struct Plan {
    int p = 0; double theta = 0.77;
    std::vector<double> pos;  // copy of input positions (N x 3)
    Tree T; Lists Ls;
};

// Reading S3: a pair at zero distance contributes nothing (eq. (3) is singular there).  rule = 0: zero distance
// means r^2 == 0 in fp64.  rule = 1 ("fp32 rule", used when the inputs are fp32 and the result is compared with the fp32 CUDA
// path): the decision is taken in the kernel's precision -- r^2 is formed in IEEE binary32 exactly as the fp32 kernels form it,
// fma(dz, dz, fma(dy, dy, dx*dx)) from the binary32 differences, and every pair with r^2 below FLT_MIN (the smallest normal
// binary32 number; |r| < 1.08e-19) counts as coincident: its 1/r^3 is not representable in binary32 anyway.
inline bool coincident(int rule, double dx, double dy, double dz) {
    if (rule == 0) return dx * dx + dy * dy + dz * dz == 0.0;
    const float fx = (float)dx, fy = (float)dy, fz = (float)dz;  // exact: differences of binary32 inputs that close are binary32 numbers
    const float r2 = std::fmaf(fz, fz, std::fmaf(fy, fy, fx * fx));
    return r2 < FLT_MIN;
}

// -------------------------------------------------------------------------------------
// Evaluate, stage order PAPER.md:251; steps E1-E7 of DESIGN.md.  If leaf_mask != nullptr only
// the leaves with mask != 0 get results (all other outputs are left untouched): local
// expansions are then computed only for those leaves and their ancestors, with the
// same arithmetic and order as the full run, so sampled outputs equal the full ones.
// -------------------------------------------------------------------------------------
void evaluate(const Plan& P, const double* q, const uint8_t* leaf_mask, double* pot, double* field, int rule = 0) {
    const Tree& T = P.T; const Lists& Ls = P.Ls;
    const int p = P.p, K = (p + 1) * (p + 1), s = T.s, L = T.L;
    const int64_t nb = T.level_off[L + 1], n_leaves = (int64_t)1 << (s * L), nch = (int64_t)1 << s;
    const int64_t leaf0 = T.level_off[L];
    const double* pos = P.pos.data();
    std::vector<double> C((size_t)nb * K, 0.0), D((size_t)nb * K, 0.0);
    std::vector<uint8_t> need(nb, leaf_mask ? 0 : 1);
    if (leaf_mask) {
        for (int64_t t = 0; t < n_leaves; ++t) if (leaf_mask[t]) need[leaf0 + t] = 1;
        for (int l = L; l >= 1; --l)
            for (int64_t b = 0; b < ((int64_t)1 << (s * l)); ++b)
                if (need[T.level_off[l] + b]) need[T.level_off[l - 1] + b / nch] = 1;
    }
    // E1: P2M at leaves, eq. (13)
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < n_leaves; ++t) {
        const int64_t g = leaf0 + t;
        std::vector<double> R(K);
        for (int64_t k = T.box_start[g]; k < T.box_start[g] + T.box_count[g]; ++k) {
            const int64_t i = T.perm[k];
            regular_basis(p, pos[3 * i] - T.ctr[3 * g], pos[3 * i + 1] - T.ctr[3 * g + 1], pos[3 * i + 2] - T.ctr[3 * g + 2], R.data());
            for (int c = 0; c < K; ++c) C[(size_t)g * K + c] += q[i] * R[c];
        }
    }
    // E2: M2M, l = L..1, children in ascending order; b = child centre - parent centre
    for (int l = L; l >= 1; --l) {
        const int64_t nbp = (int64_t)1 << (s * (l - 1));
#pragma omp parallel for schedule(dynamic, 4)
        for (int64_t bp = 0; bp < nbp; ++bp) {
            const int64_t gp = T.level_off[l - 1] + bp;
            std::vector<double> tmp(K);
            for (int64_t j = 0; j < nch; ++j) {
                const int64_t gc = T.level_off[l] + bp * nch + j;
                if (T.box_count[gc] == 0) continue;
                const double b[3] = {T.ctr[3 * gc] - T.ctr[3 * gp], T.ctr[3 * gc + 1] - T.ctr[3 * gp + 1], T.ctr[3 * gc + 2] - T.ctr[3 * gp + 2]};
                translate(0, p, &C[(size_t)gc * K], b, tmp.data());
                for (int c = 0; c < K; ++c) C[(size_t)gp * K + c] += tmp[c];
            }
        }
    }
    // E3: M2L over the weak list, all levels; b = source centre - target centre
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t gt = 0; gt < nb; ++gt) {
        if (!need[gt]) continue;
        std::vector<double> tmp(K);
        for (int64_t e = Ls.weak_off[gt]; e < Ls.weak_off[gt + 1]; ++e) {
            const int64_t gs = Ls.weak_src[e];
            const double b[3] = {T.ctr[3 * gs] - T.ctr[3 * gt], T.ctr[3 * gs + 1] - T.ctr[3 * gt + 1], T.ctr[3 * gs + 2] - T.ctr[3 * gt + 2]};
            translate(1, p, &C[(size_t)gs * K], b, tmp.data());
            for (int c = 0; c < K; ++c) D[(size_t)gt * K + c] += tmp[c];
        }
    }
    // E4: L2L, l = 1..L; b = parent centre - child centre
    for (int l = 1; l <= L; ++l) {
        const int64_t nbl = (int64_t)1 << (s * l);
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t bc = 0; bc < nbl; ++bc) {
            const int64_t gc = T.level_off[l] + bc, gp = T.level_off[l - 1] + bc / nch;
            if (!need[gc] || T.box_count[gc] == 0) continue;
            std::vector<double> tmp(K);
            const double b[3] = {T.ctr[3 * gp] - T.ctr[3 * gc], T.ctr[3 * gp + 1] - T.ctr[3 * gc + 1], T.ctr[3 * gp + 2] - T.ctr[3 * gc + 2]};
            translate(2, p, &D[(size_t)gp * K], b, tmp.data());
            for (int c = 0; c < K; ++c) D[(size_t)gc * K + c] += tmp[c];
        }
    }
    // E5 L2P (eq. 14, gradient App. A.3), E6 P2P, E7 scaling and scatter
    const double inv4pi = 1.0 / (4.0 * M_PI);
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t t = 0; t < n_leaves; ++t) {
        if (leaf_mask && !leaf_mask[t]) continue;
        const int64_t g = leaf0 + t;
        std::vector<double> R(K), G(3 * K);
        for (int64_t k = T.box_start[g]; k < T.box_start[g] + T.box_count[g]; ++k) {
            const int64_t i = T.perm[k];
            const double x = pos[3 * i] - T.ctr[3 * g], y = pos[3 * i + 1] - T.ctr[3 * g + 1], z = pos[3 * i + 2] - T.ctr[3 * g + 2];
            regular_basis(p, x, y, z, R.data());
            regular_grad(p, x, y, z, R.data(), G.data());
            double phi_far = 0.0, gfar[3] = {0, 0, 0};
            for (int n = 0; n <= p; ++n)
                for (int m = -n; m <= n; ++m) {
                    const double w = ((m == 0) ? 1.0 : 2.0) * sgn(m) * D[(size_t)g * K + IDX(n, m)];
                    phi_far += w * R[IDX(n, m)];
                    for (int c = 0; c < 3; ++c) gfar[c] += w * G[3 * IDX(n, m) + c];
                }
            double phi_near = 0.0, gnear[3] = {0, 0, 0};
            for (int64_t e = Ls.strong_off[t]; e < Ls.strong_off[t + 1]; ++e) {
                const int64_t gs = leaf0 + Ls.strong_src[e];
                for (int64_t kk = T.box_start[gs]; kk < T.box_start[gs] + T.box_count[gs]; ++kk) {
                    const int64_t j = T.perm[kk];
                    if (j == i) continue;  // S3
                    const double dx = pos[3 * i] - pos[3 * j], dy = pos[3 * i + 1] - pos[3 * j + 1], dz = pos[3 * i + 2] - pos[3 * j + 2];
                    if (coincident(rule, dx, dy, dz)) continue;  // S3: coincident points contribute nothing
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    const double r = std::sqrt(r2);
                    phi_near += q[j] / r;
                    const double f = q[j] / (r2 * r);
                    gnear[0] -= f * dx; gnear[1] -= f * dy; gnear[2] -= f * dz;
                }
            }
            if (pot) pot[i] = -(phi_far + phi_near) * inv4pi;  // eqs. (2),(9),(14)
            if (field) for (int c = 0; c < 3; ++c) field[3 * i + c] = (gfar[c] + gnear[c]) * inv4pi;  // field = -grad u (S2)
        }
    }
}

// -------------------------------------------------------------------------------------
// Separate sources and targets: one hierarchy over the source points, one over the target points
// (same rules T1-T7, same N_max and s), interaction lists by level marching over the two hierarchies, evaluate =
// P2M/M2M on the source hierarchy, M2L across, L2L/L2P on the target hierarchy, P2P between target and source leaves.
// -------------------------------------------------------------------------------------
// eq. (4) between a target box and a source box; the same expression and evaluation order as admissible()
bool admissible_st(const Tree& Tt, int64_t gt, const Tree& Ts, int64_t gs, double theta) {
    const double ra = Tt.rad[gt], rb = Ts.rad[gs];
    const double R = std::max(ra, rb), r = std::min(ra, rb);
    const double dx = Tt.ctr[3 * gt] - Ts.ctr[3 * gs], dy = Tt.ctr[3 * gt + 1] - Ts.ctr[3 * gs + 1], dz = Tt.ctr[3 * gt + 2] - Ts.ctr[3 * gs + 2];
    const double d = std::sqrt((dx * dx + dy * dy) + dz * dz);
    return R + theta * r < theta * d;
}
// "average box radius" of a level: mean of the radii of its non-empty boxes, summed in box order
double mean_radius(const Tree& T, int l) {
    double sum = 0.0; int64_t cnt = 0;
    for (int64_t b = 0; b < ((int64_t)1 << (T.s * l)); ++b) {
        const int64_t g = T.level_off[l] + b;
        if (T.box_count[g] > 0) { sum += T.rad[g]; ++cnt; }
    }
    return cnt ? sum / (double)cnt : 0.0;
}
// Level marching, started at (l_trg, l_src) = (0, 0): 1. increase the level with the larger average box
// radius; 2. if equal, the source level; 3. if one hierarchy has no more levels, the other; 4. stop when no pair is left
// or both are at their leaf level.  Weak rows: per target box (global id in Tt) the source boxes (global ids in Ts),
// ascending; strong rows: per target leaf the source leaves still failing at (L_trg, L_src).  steps: the (l_trg, l_src) visited.
void build_lists_st(const Tree& Tt, const Tree& Ts, double theta, Lists& Ls, std::vector<int>& steps) {
    const int s = Tt.s, Lt = Tt.L, Lsrc = Ts.L;
    const int64_t nch = (int64_t)1 << s;
    const int64_t nbt = Tt.level_off[Lt + 1];
    const int64_t n_tleaves = (int64_t)1 << (s * Lt);
    std::vector<std::vector<int64_t>> weak_rows(nbt), strong_rows(n_tleaves);
    std::vector<std::pair<int64_t, int64_t>> cand, fail;
    cand.push_back({0, 0});
    int lt = 0, ls = 0;
    steps.clear();
    for (;;) {
        steps.push_back(lt); steps.push_back(ls);
        fail.clear();
        for (auto& pr : cand) {
            const int64_t gt = Tt.level_off[lt] + pr.first, gs = Ts.level_off[ls] + pr.second;
            if (admissible_st(Tt, gt, Ts, gs, theta)) weak_rows[gt].push_back(gs);
            else fail.push_back(pr);
        }
        if (lt == Lt && ls == Lsrc) break;
        bool refine_src;
        if (ls == Lsrc) refine_src = false;            // rule 3
        else if (lt == Lt) refine_src = true;          // rule 3
        else refine_src = !(mean_radius(Tt, lt) > mean_radius(Ts, ls));  // rules 1, 2
        cand.clear();
        for (auto& pr : fail)
            for (int64_t c = 0; c < nch; ++c) {
                const int64_t a = refine_src ? pr.first : pr.first * nch + c, b = refine_src ? pr.second * nch + c : pr.second;
                if (Tt.box_count[Tt.level_off[lt + (refine_src ? 0 : 1)] + a] == 0 || Ts.box_count[Ts.level_off[ls + (refine_src ? 1 : 0)] + b] == 0)
                    continue;  // T5
                cand.push_back({a, b});
            }
        if (refine_src) ++ls; else ++lt;
    }
    for (auto& pr : fail) strong_rows[pr.first].push_back(pr.second);
    Ls.weak_off.assign(nbt + 1, 0); Ls.weak_src.clear();
    for (int64_t g = 0; g < nbt; ++g) {
        std::sort(weak_rows[g].begin(), weak_rows[g].end());
        for (int64_t v : weak_rows[g]) Ls.weak_src.push_back(v);
        Ls.weak_off[g + 1] = (int64_t)Ls.weak_src.size();
    }
    Ls.strong_off.assign(n_tleaves + 1, 0); Ls.strong_src.clear();
    for (int64_t t = 0; t < n_tleaves; ++t) {
        std::sort(strong_rows[t].begin(), strong_rows[t].end());
        for (int64_t v : strong_rows[t]) Ls.strong_src.push_back(v);
        Ls.strong_off[t + 1] = (int64_t)Ls.strong_src.size();
    }
}

struct PlanST {
    int p = 0; double theta = 0.77;
    std::vector<double> spos, tpos;
    Tree Ts, Tt; Lists Ls;
    std::vector<int> steps;
};

// potential and field at the targets from charges q at the sources; steps E1-E7 with the two hierarchies.  leaf_mask (target
// leaves) works as in evaluate(): only the masked leaves get results, computed with the same arithmetic as in a full run.
void evaluate_st(const PlanST& P, const double* q, const uint8_t* leaf_mask, double* pot, double* field, int rule = 0) {
    const Tree& Ts = P.Ts; const Tree& Tt = P.Tt; const Lists& Ls = P.Ls;
    const int p = P.p, K = (p + 1) * (p + 1), s = Ts.s;
    const int64_t nch = (int64_t)1 << s;
    const int64_t nbs = Ts.level_off[Ts.L + 1], nbt = Tt.level_off[Tt.L + 1];
    const int64_t n_sleaves = (int64_t)1 << (s * Ts.L), n_tleaves = (int64_t)1 << (s * Tt.L);
    const int64_t sleaf0 = Ts.level_off[Ts.L], tleaf0 = Tt.level_off[Tt.L];
    const double* spos = P.spos.data(); const double* tpos = P.tpos.data();
    std::vector<double> C((size_t)nbs * K, 0.0), D((size_t)nbt * K, 0.0);
    std::vector<uint8_t> need(nbt, leaf_mask ? 0 : 1);
    if (leaf_mask) {
        for (int64_t t = 0; t < n_tleaves; ++t) if (leaf_mask[t]) need[tleaf0 + t] = 1;
        for (int l = Tt.L; l >= 1; --l)
            for (int64_t b = 0; b < ((int64_t)1 << (s * l)); ++b)
                if (need[Tt.level_off[l] + b]) need[Tt.level_off[l - 1] + b / nch] = 1;
    }
    // E1: P2M at the source leaves, eq. (13)
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < n_sleaves; ++t) {
        const int64_t g = sleaf0 + t;
        std::vector<double> R(K);
        for (int64_t k = Ts.box_start[g]; k < Ts.box_start[g] + Ts.box_count[g]; ++k) {
            const int64_t i = Ts.perm[k];
            regular_basis(p, spos[3 * i] - Ts.ctr[3 * g], spos[3 * i + 1] - Ts.ctr[3 * g + 1], spos[3 * i + 2] - Ts.ctr[3 * g + 2], R.data());
            for (int c = 0; c < K; ++c) C[(size_t)g * K + c] += q[i] * R[c];
        }
    }
    // E2: M2M in the source hierarchy; b = child centre - parent centre
    for (int l = Ts.L; l >= 1; --l) {
        const int64_t nbp = (int64_t)1 << (s * (l - 1));
#pragma omp parallel for schedule(dynamic, 4)
        for (int64_t bp = 0; bp < nbp; ++bp) {
            const int64_t gp = Ts.level_off[l - 1] + bp;
            std::vector<double> tmp(K);
            for (int64_t j = 0; j < nch; ++j) {
                const int64_t gc = Ts.level_off[l] + bp * nch + j;
                if (Ts.box_count[gc] == 0) continue;
                const double b[3] = {Ts.ctr[3 * gc] - Ts.ctr[3 * gp], Ts.ctr[3 * gc + 1] - Ts.ctr[3 * gp + 1], Ts.ctr[3 * gc + 2] - Ts.ctr[3 * gp + 2]};
                translate(0, p, &C[(size_t)gc * K], b, tmp.data());
                for (int c = 0; c < K; ++c) C[(size_t)gp * K + c] += tmp[c];
            }
        }
    }
    // E3: M2L over the weak list; b = source centre - target centre
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t gt = 0; gt < nbt; ++gt) {
        if (!need[gt]) continue;
        std::vector<double> tmp(K);
        for (int64_t e = Ls.weak_off[gt]; e < Ls.weak_off[gt + 1]; ++e) {
            const int64_t gs = Ls.weak_src[e];
            const double b[3] = {Ts.ctr[3 * gs] - Tt.ctr[3 * gt], Ts.ctr[3 * gs + 1] - Tt.ctr[3 * gt + 1], Ts.ctr[3 * gs + 2] - Tt.ctr[3 * gt + 2]};
            translate(1, p, &C[(size_t)gs * K], b, tmp.data());
            for (int c = 0; c < K; ++c) D[(size_t)gt * K + c] += tmp[c];
        }
    }
    // E4: L2L in the target hierarchy; b = parent centre - child centre
    for (int l = 1; l <= Tt.L; ++l) {
        const int64_t nbl = (int64_t)1 << (s * l);
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t bc = 0; bc < nbl; ++bc) {
            const int64_t gc = Tt.level_off[l] + bc, gp = Tt.level_off[l - 1] + bc / nch;
            if (!need[gc] || Tt.box_count[gc] == 0) continue;
            std::vector<double> tmp(K);
            const double b[3] = {Tt.ctr[3 * gp] - Tt.ctr[3 * gc], Tt.ctr[3 * gp + 1] - Tt.ctr[3 * gc + 1], Tt.ctr[3 * gp + 2] - Tt.ctr[3 * gc + 2]};
            translate(2, p, &D[(size_t)gp * K], b, tmp.data());
            for (int c = 0; c < K; ++c) D[(size_t)gc * K + c] += tmp[c];
        }
    }
    // E5 L2P, E6 P2P (every source of the strong-listed source leaves; zero-distance pairs contribute nothing, S3), E7
    const double inv4pi = 1.0 / (4.0 * M_PI);
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t t = 0; t < n_tleaves; ++t) {
        if (leaf_mask && !leaf_mask[t]) continue;
        const int64_t g = tleaf0 + t;
        std::vector<double> R(K), G(3 * K);
        for (int64_t k = Tt.box_start[g]; k < Tt.box_start[g] + Tt.box_count[g]; ++k) {
            const int64_t i = Tt.perm[k];
            const double x = tpos[3 * i] - Tt.ctr[3 * g], y = tpos[3 * i + 1] - Tt.ctr[3 * g + 1], z = tpos[3 * i + 2] - Tt.ctr[3 * g + 2];
            regular_basis(p, x, y, z, R.data());
            regular_grad(p, x, y, z, R.data(), G.data());
            double phi_far = 0.0, gfar[3] = {0, 0, 0};
            for (int n = 0; n <= p; ++n)
                for (int m = -n; m <= n; ++m) {
                    const double w = ((m == 0) ? 1.0 : 2.0) * sgn(m) * D[(size_t)g * K + IDX(n, m)];
                    phi_far += w * R[IDX(n, m)];
                    for (int c = 0; c < 3; ++c) gfar[c] += w * G[3 * IDX(n, m) + c];
                }
            double phi_near = 0.0, gnear[3] = {0, 0, 0};
            for (int64_t e = Ls.strong_off[t]; e < Ls.strong_off[t + 1]; ++e) {
                const int64_t gs = sleaf0 + Ls.strong_src[e];
                for (int64_t kk = Ts.box_start[gs]; kk < Ts.box_start[gs] + Ts.box_count[gs]; ++kk) {
                    const int64_t j = Ts.perm[kk];
                    const double dx = tpos[3 * i] - spos[3 * j], dy = tpos[3 * i + 1] - spos[3 * j + 1], dz = tpos[3 * i + 2] - spos[3 * j + 2];
                    if (coincident(rule, dx, dy, dz)) continue;  // S3
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    const double r = std::sqrt(r2);
                    phi_near += q[j] / r;
                    const double f = q[j] / (r2 * r);
                    gnear[0] -= f * dx; gnear[1] -= f * dy; gnear[2] -= f * dz;
                }
            }
            if (pot) pot[i] = -(phi_far + phi_near) * inv4pi;
            if (field) for (int c = 0; c < 3; ++c) field[3 * i + c] = (gfar[c] + gnear[c]) * inv4pi;
        }
    }
}


// -------------------------------------------------------------------------------------
// Adjoint evaluate.  The paper differentiates eval_potential with respect to the charges by JAX autodiff;
// the evaluate is linear in q -- potential = A q, field = F q with the FMM operators A, F of evaluate() / evaluate_st() -- so the
// vector-Jacobian product autodiff returns for cotangents (ubar, fbar) is  qbar = A^T ubar + F^T fbar:  every step E1-E7
// transposed and run in reverse order.  Nothing clever: the transposed translation operators are formed literally, column k of
// T = translate(e_k), and applied as T^T x.  Tt / tpos: hierarchy and points of the targets, Ts / spos: of the sources (the same
// objects for a single point set, where the pair i == j is excluded as in evaluate()).
// -------------------------------------------------------------------------------------
void translate_transposed(int kind, int p, const double* in, const double b[3], double* out) {
    const int K = (p + 1) * (p + 1);
    std::vector<double> e(K, 0.0), col(K);
    for (int k = 0; k < K; ++k) {
        e[k] = 1.0;
        translate(kind, p, e.data(), b, col.data());  // column k of T
        e[k] = 0.0;
        double acc = 0.0;
        for (int c = 0; c < K; ++c) acc += col[c] * in[c];
        out[k] = acc;  // (T^T in)_k = sum_c T[c][k] in[c]
    }
}

void adjoint_impl(int p, const Tree& Tt, const double* tpos, const Tree& Ts, const double* spos, const Lists& Ls, bool same_set,
                  const double* ubar, const double* fbar, double* qbar, int rule) {
    const int K = (p + 1) * (p + 1), s = Ts.s;
    const int64_t nch = (int64_t)1 << s;
    const int64_t nbs = Ts.level_off[Ts.L + 1], nbt = Tt.level_off[Tt.L + 1];
    const int64_t n_sleaves = (int64_t)1 << (s * Ts.L), n_tleaves = (int64_t)1 << (s * Tt.L);
    const int64_t sleaf0 = Ts.level_off[Ts.L], tleaf0 = Tt.level_off[Tt.L];
    const int64_t Ns = (int64_t)Ts.perm.size();
    const double inv4pi = 1.0 / (4.0 * M_PI);
    std::vector<double> Cbar((size_t)nbs * K, 0.0), Dbar((size_t)nbt * K, 0.0);
    for (int64_t j = 0; j < Ns; ++j) qbar[j] = 0.0;
    // E7^T: u = -(phi_far + phi_near)/4pi, field = (g_far + g_near)/4pi  =>  phibar = -ubar/4pi, gbar = fbar/4pi (both parts)
    // E6^T (P2P) and E5^T (L2P), target leaf by target leaf (serial: the P2P part scatters into the sources)
    for (int64_t t = 0; t < n_tleaves; ++t) {
        const int64_t g = tleaf0 + t;
        std::vector<double> R(K), G(3 * K);
        for (int64_t k = Tt.box_start[g]; k < Tt.box_start[g] + Tt.box_count[g]; ++k) {
            const int64_t i = Tt.perm[k];
            const double phibar = ubar ? -ubar[i] * inv4pi : 0.0;
            const double gbar[3] = {fbar ? fbar[3 * i] * inv4pi : 0.0, fbar ? fbar[3 * i + 1] * inv4pi : 0.0, fbar ? fbar[3 * i + 2] * inv4pi : 0.0};
            const double x = tpos[3 * i] - Tt.ctr[3 * g], y = tpos[3 * i + 1] - Tt.ctr[3 * g + 1], z = tpos[3 * i + 2] - Tt.ctr[3 * g + 2];
            regular_basis(p, x, y, z, R.data());
            regular_grad(p, x, y, z, R.data(), G.data());
            // E5^T: phi_far = sum w D R, g_far = sum w D G   =>   Dbar += w (phibar R + gbar . G)
            for (int n = 0; n <= p; ++n)
                for (int m = -n; m <= n; ++m) {
                    const double w = ((m == 0) ? 1.0 : 2.0) * sgn(m);
                    const int c = IDX(n, m);
                    Dbar[(size_t)g * K + c] += w * (phibar * R[c] + gbar[0] * G[3 * c] + gbar[1] * G[3 * c + 1] + gbar[2] * G[3 * c + 2]);
                }
            // E6^T: phi_near += q_j / r, g_near -= q_j d / r^3   =>   qbar_j += phibar / r - (gbar . d) / r^3
            for (int64_t e = Ls.strong_off[t]; e < Ls.strong_off[t + 1]; ++e) {
                const int64_t gs = sleaf0 + Ls.strong_src[e];
                for (int64_t kk = Ts.box_start[gs]; kk < Ts.box_start[gs] + Ts.box_count[gs]; ++kk) {
                    const int64_t j = Ts.perm[kk];
                    if (same_set && j == i) continue;  // S3
                    const double dx = tpos[3 * i] - spos[3 * j], dy = tpos[3 * i + 1] - spos[3 * j + 1], dz = tpos[3 * i + 2] - spos[3 * j + 2];
                    if (coincident(rule, dx, dy, dz)) continue;  // S3
                    const double r2 = dx * dx + dy * dy + dz * dz;
                    const double r = std::sqrt(r2);
                    qbar[j] += phibar / r - (gbar[0] * dx + gbar[1] * dy + gbar[2] * dz) / (r2 * r);
                }
            }
        }
    }
    // E4^T: D_child += T_L2L(b = parent - child) D_parent for l = 1..L   =>   Dbar_parent += T^T Dbar_child, l = L..1
    for (int l = Tt.L; l >= 1; --l) {
        const int64_t nbp = (int64_t)1 << (s * (l - 1));
#pragma omp parallel for schedule(dynamic, 4)
        for (int64_t bp = 0; bp < nbp; ++bp) {
            const int64_t gp = Tt.level_off[l - 1] + bp;
            std::vector<double> tmp(K);
            for (int64_t j = 0; j < nch; ++j) {
                const int64_t gc = Tt.level_off[l] + bp * nch + j;
                if (Tt.box_count[gc] == 0) continue;
                const double b[3] = {Tt.ctr[3 * gp] - Tt.ctr[3 * gc], Tt.ctr[3 * gp + 1] - Tt.ctr[3 * gc + 1], Tt.ctr[3 * gp + 2] - Tt.ctr[3 * gc + 2]};
                translate_transposed(2, p, &Dbar[(size_t)gc * K], b, tmp.data());
                for (int c = 0; c < K; ++c) Dbar[(size_t)gp * K + c] += tmp[c];
            }
        }
    }
    // E3^T: D_t += T_M2L(b = c_s - c_t) C_s over the weak list   =>   Cbar_s += T^T Dbar_t.  Rows of the transposed list (by
    // source box) are independent, so the loop runs over sources; targets of a source in ascending order.
    {
        std::vector<std::vector<int64_t>> by_src(nbs);
        for (int64_t gt = 0; gt < nbt; ++gt)
            for (int64_t e = Ls.weak_off[gt]; e < Ls.weak_off[gt + 1]; ++e) by_src[Ls.weak_src[e]].push_back(gt);
#pragma omp parallel for schedule(dynamic, 4)
        for (int64_t gs = 0; gs < nbs; ++gs) {
            std::vector<double> tmp(K);
            for (int64_t gt : by_src[gs]) {
                const double b[3] = {Ts.ctr[3 * gs] - Tt.ctr[3 * gt], Ts.ctr[3 * gs + 1] - Tt.ctr[3 * gt + 1], Ts.ctr[3 * gs + 2] - Tt.ctr[3 * gt + 2]};
                translate_transposed(1, p, &Dbar[(size_t)gt * K], b, tmp.data());
                for (int c = 0; c < K; ++c) Cbar[(size_t)gs * K + c] += tmp[c];
            }
        }
    }
    // E2^T: C_parent += T_M2M(b = child - parent) C_child for l = L..1   =>   Cbar_child += T^T Cbar_parent, l = 1..L
    for (int l = 1; l <= Ts.L; ++l) {
        const int64_t nbl = (int64_t)1 << (s * l);
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t bc = 0; bc < nbl; ++bc) {
            const int64_t gc = Ts.level_off[l] + bc, gp = Ts.level_off[l - 1] + bc / nch;
            if (Ts.box_count[gc] == 0) continue;
            std::vector<double> tmp(K);
            const double b[3] = {Ts.ctr[3 * gc] - Ts.ctr[3 * gp], Ts.ctr[3 * gc + 1] - Ts.ctr[3 * gp + 1], Ts.ctr[3 * gc + 2] - Ts.ctr[3 * gp + 2]};
            translate_transposed(0, p, &Cbar[(size_t)gp * K], b, tmp.data());
            for (int c = 0; c < K; ++c) Cbar[(size_t)gc * K + c] += tmp[c];
        }
    }
    // E1^T: C_leaf += q_i R^(r_i - c)   =>   qbar_i += sum_c Cbar_leaf[c] R^_c(r_i - c)
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t t = 0; t < n_sleaves; ++t) {
        const int64_t g = sleaf0 + t;
        std::vector<double> R(K);
        for (int64_t k = Ts.box_start[g]; k < Ts.box_start[g] + Ts.box_count[g]; ++k) {
            const int64_t i = Ts.perm[k];
            regular_basis(p, spos[3 * i] - Ts.ctr[3 * g], spos[3 * i + 1] - Ts.ctr[3 * g + 1], spos[3 * i + 2] - Ts.ctr[3 * g + 2], R.data());
            double acc = 0.0;
            for (int c = 0; c < K; ++c) acc += Cbar[(size_t)g * K + c] * R[c];
            qbar[i] += acc;
        }
    }
}

}  // namespace

// =====================================================================================
// C interface for ctypes (tests, smoke, bench cpu_baseline).  All pointers are host.
// =====================================================================================
extern "C" {

void orc_regular_basis(int p, double x, double y, double z, double* R) { regular_basis(p, x, y, z, R); }
void orc_singular_basis(int p, double x, double y, double z, double* S) { singular_basis(p, x, y, z, S); }
void orc_regular_grad(int p, double x, double y, double z, double* G) {
    std::vector<double> R((p + 1) * (p + 1));
    regular_basis(p, x, y, z, R.data());
    regular_grad(p, x, y, z, R.data(), G);
}
double orc_wigner_d(int j, int mp, int m, double beta) { return wigner_d(j, mp, m, beta); }
void orc_rot_azimuthal(int p, int local_type, const double* in, double dphi, double* out) { rot_azimuthal(p, local_type, in, dphi, out); }
void orc_rot_polar(int p, int local_type, const double* in, double dtheta, double* out) { rot_polar(p, local_type, in, dtheta, out); }
void orc_shift(int kind, int p, const double* in, double r, double* out) {
    if (kind == 0) shift_m2m(p, in, r, out); else if (kind == 1) shift_m2l(p, in, r, out); else shift_l2l(p, in, r, out);
}
void orc_translate(int kind, int p, const double* in, const double* b, double* out) { translate(kind, p, in, b, out); }
int orc_tree_depth(int64_t N, int N_max, int s) { return tree_depth(N, N_max, s); }

void* orc_plan_create(const double* pos, int64_t N, int p, int N_max, int s, double theta, int cross_level) {
    Plan* P = new Plan();
    P->p = p; P->theta = theta;
    P->pos.assign(pos, pos + 3 * N);
    build_tree(P->pos.data(), N, N_max, s, P->T);
    build_lists(P->T, theta, P->Ls, cross_level);
    return P;
}
void orc_plan_destroy(void* h) { delete (Plan*)h; }
void orc_plan_info(void* h, int* L, int64_t* n_boxes, int64_t* n_leaves, int64_t* n_weak, int64_t* n_strong, int64_t* n_p2p_pairs) {
    Plan* P = (Plan*)h;
    *L = P->T.L; *n_boxes = P->T.level_off[P->T.L + 1]; *n_leaves = (int64_t)1 << (P->T.s * P->T.L);
    *n_weak = (int64_t)P->Ls.weak_src.size(); *n_strong = (int64_t)P->Ls.strong_src.size();
    int64_t pairs = 0;
    const int64_t leaf0 = P->T.level_off[P->T.L];
    for (int64_t t = 0; t < *n_leaves; ++t)
        for (int64_t e = P->Ls.strong_off[t]; e < P->Ls.strong_off[t + 1]; ++e)
            pairs += P->T.box_count[leaf0 + t] * P->T.box_count[leaf0 + P->Ls.strong_src[e]];
    *n_p2p_pairs = pairs;
}
void orc_plan_copy_tree(void* h, int64_t* perm, int64_t* box_start, int64_t* box_count, double* lo, double* hi, double* ctr, double* rad) {
    Plan* P = (Plan*)h; const Tree& T = P->T;
    const int64_t nb = T.level_off[T.L + 1];
    if (perm) std::copy(T.perm.begin(), T.perm.end(), perm);
    if (box_start) std::copy(T.box_start.begin(), T.box_start.end(), box_start);
    if (box_count) std::copy(T.box_count.begin(), T.box_count.end(), box_count);
    if (lo) std::copy(T.lo.begin(), T.lo.begin() + 3 * nb, lo);
    if (hi) std::copy(T.hi.begin(), T.hi.begin() + 3 * nb, hi);
    if (ctr) std::copy(T.ctr.begin(), T.ctr.begin() + 3 * nb, ctr);
    if (rad) std::copy(T.rad.begin(), T.rad.begin() + nb, rad);
}
void orc_plan_copy_lists(void* h, int64_t* weak_off, int64_t* weak_src, int64_t* strong_off, int64_t* strong_src) {
    Plan* P = (Plan*)h; const Lists& Ls = P->Ls;
    if (weak_off) std::copy(Ls.weak_off.begin(), Ls.weak_off.end(), weak_off);
    if (weak_src) std::copy(Ls.weak_src.begin(), Ls.weak_src.end(), weak_src);
    if (strong_off) std::copy(Ls.strong_off.begin(), Ls.strong_off.end(), strong_off);
    if (strong_src) std::copy(Ls.strong_src.begin(), Ls.strong_src.end(), strong_src);
}
// lists from hand-made geometry (pin PAPER.md:80): boxes given by ctr/rad, tree shape (s, L) complete
void orc_lists_from_geometry(int s, int L, const double* ctr, const double* rad, double theta, int cross_level,
                             int64_t* n_weak_per_box, int64_t* n_strong_per_leaf) {
    Tree T; T.s = s; T.L = L;
    T.level_off.assign(L + 2, 0);
    for (int l = 0; l <= L; ++l) T.level_off[l + 1] = T.level_off[l] + ((int64_t)1 << (s * l));
    const int64_t nb = T.level_off[L + 1];
    T.ctr.assign(ctr, ctr + 3 * nb); T.rad.assign(rad, rad + nb);
    T.box_count.assign(nb, 1); T.box_start.assign(nb, 0);
    Lists Ls; build_lists(T, theta, Ls, cross_level);
    for (int64_t g = 0; g < nb; ++g) n_weak_per_box[g] = Ls.weak_off[g + 1] - Ls.weak_off[g];
    const int64_t nl = (int64_t)1 << (s * L);
    for (int64_t t = 0; t < nl; ++t) n_strong_per_leaf[t] = Ls.strong_off[t + 1] - Ls.strong_off[t];
}
void orc_evaluate(void* h, const double* q, const uint8_t* leaf_mask, double* pot, double* field, int rule) {
    evaluate(*(Plan*)h, q, leaf_mask, pot, field, rule);
}
// qbar (N) = A^T ubar + F^T fbar for the FMM operators of orc_evaluate (ubar: N or NULL, fbar: N x 3 or NULL)
void orc_evaluate_adjoint(void* h, const double* ubar, const double* fbar, double* qbar, int rule) {
    Plan* P = (Plan*)h;
    adjoint_impl(P->p, P->T, P->pos.data(), P->T, P->pos.data(), P->Ls, true, ubar, fbar, qbar, rule);
}
// plain definition, eqs. (1)-(3) PAPER.md:19-28: u_i = -(1/4pi) sum_{j != i} q_j/|r_i - r_j|, field = -grad u;
// evaluated at the targets listed in tgt (indices into pos), against all N sources.
void orc_direct(const double* pos, const double* q, int64_t N, const int64_t* tgt, int64_t n_tgt, double* pot, double* field, int rule) {
    const double inv4pi = 1.0 / (4.0 * M_PI);
#pragma omp parallel for schedule(static)
    for (int64_t a = 0; a < n_tgt; ++a) {
        const int64_t i = tgt[a];
        double ph = 0.0, g[3] = {0, 0, 0};
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            const double dx = pos[3 * i] - pos[3 * j], dy = pos[3 * i + 1] - pos[3 * j + 1], dz = pos[3 * i + 2] - pos[3 * j + 2];
            if (coincident(rule, dx, dy, dz)) continue;
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double r = std::sqrt(r2);
            ph += q[j] / r;
            const double f = q[j] / (r2 * r);
            g[0] -= f * dx; g[1] -= f * dy; g[2] -= f * dz;
        }
        if (pot) pot[a] = -ph * inv4pi;
        if (field) for (int c = 0; c < 3; ++c) field[3 * a + c] = g[c] * inv4pi;
    }
}
// ---- separate sources and targets
void* orc_plan_st_create(const double* spos, int64_t Ns, const double* tpos, int64_t Nt, int p, int N_max, int s, double theta) {
    PlanST* P = new PlanST();
    P->p = p; P->theta = theta;
    P->spos.assign(spos, spos + 3 * Ns); P->tpos.assign(tpos, tpos + 3 * Nt);
    build_tree(P->spos.data(), Ns, N_max, s, P->Ts);
    build_tree(P->tpos.data(), Nt, N_max, s, P->Tt);
    build_lists_st(P->Tt, P->Ts, theta, P->Ls, P->steps);
    return P;
}
void orc_plan_st_destroy(void* h) { delete (PlanST*)h; }
// which: 0 = source hierarchy, 1 = target hierarchy
void orc_plan_st_info(void* h, int which, int* L, int64_t* n_boxes, int64_t* n_leaves, int64_t* n_weak, int64_t* n_strong, int64_t* n_p2p_pairs, int* n_steps) {
    PlanST* P = (PlanST*)h; const Tree& T = which ? P->Tt : P->Ts;
    *L = T.L; *n_boxes = T.level_off[T.L + 1]; *n_leaves = (int64_t)1 << (T.s * T.L);
    *n_weak = (int64_t)P->Ls.weak_src.size(); *n_strong = (int64_t)P->Ls.strong_src.size();
    int64_t pairs = 0;
    const int64_t tleaf0 = P->Tt.level_off[P->Tt.L], sleaf0 = P->Ts.level_off[P->Ts.L];
    for (int64_t t = 0; t < ((int64_t)1 << (P->Tt.s * P->Tt.L)); ++t)
        for (int64_t e = P->Ls.strong_off[t]; e < P->Ls.strong_off[t + 1]; ++e)
            pairs += P->Tt.box_count[tleaf0 + t] * P->Ts.box_count[sleaf0 + P->Ls.strong_src[e]];
    *n_p2p_pairs = pairs;
    *n_steps = (int)(P->steps.size() / 2);
}
void orc_plan_st_copy_tree(void* h, int which, int64_t* perm, int64_t* box_start, int64_t* box_count, double* lo, double* hi, double* ctr, double* rad) {
    PlanST* P = (PlanST*)h; const Tree& T = which ? P->Tt : P->Ts;
    const int64_t nb = T.level_off[T.L + 1];
    if (perm) std::copy(T.perm.begin(), T.perm.end(), perm);
    if (box_start) std::copy(T.box_start.begin(), T.box_start.end(), box_start);
    if (box_count) std::copy(T.box_count.begin(), T.box_count.end(), box_count);
    if (lo) std::copy(T.lo.begin(), T.lo.begin() + 3 * nb, lo);
    if (hi) std::copy(T.hi.begin(), T.hi.begin() + 3 * nb, hi);
    if (ctr) std::copy(T.ctr.begin(), T.ctr.begin() + 3 * nb, ctr);
    if (rad) std::copy(T.rad.begin(), T.rad.begin() + nb, rad);
}
void orc_plan_st_copy_lists(void* h, int64_t* weak_off, int64_t* weak_src, int64_t* strong_off, int64_t* strong_src, int* steps) {
    PlanST* P = (PlanST*)h; const Lists& Ls = P->Ls;
    if (weak_off) std::copy(Ls.weak_off.begin(), Ls.weak_off.end(), weak_off);
    if (weak_src) std::copy(Ls.weak_src.begin(), Ls.weak_src.end(), weak_src);
    if (strong_off) std::copy(Ls.strong_off.begin(), Ls.strong_off.end(), strong_off);
    if (strong_src) std::copy(Ls.strong_src.begin(), Ls.strong_src.end(), strong_src);
    if (steps) std::copy(P->steps.begin(), P->steps.end(), steps);
}
void orc_evaluate_st(void* h, const double* q, const uint8_t* leaf_mask, double* pot, double* field, int rule) {
    evaluate_st(*(PlanST*)h, q, leaf_mask, pot, field, rule);
}
// qbar (Ns) = A^T ubar + F^T fbar for the operators of orc_evaluate_st (ubar: Nt or NULL, fbar: Nt x 3 or NULL)
void orc_evaluate_st_adjoint(void* h, const double* ubar, const double* fbar, double* qbar, int rule) {
    PlanST* P = (PlanST*)h;
    adjoint_impl(P->p, P->Tt, P->tpos.data(), P->Ts, P->spos.data(), P->Ls, false, ubar, fbar, qbar, rule);
}
// plain definition at separate targets: u(t_i) = -(1/4pi) sum_j q_j/|t_i - s_j|, field = -grad u; zero-distance pairs skipped (S3)
void orc_direct_st(const double* spos, const double* q, int64_t Ns, const double* tpos, int64_t Nt, double* pot, double* field, int rule) {
    const double inv4pi = 1.0 / (4.0 * M_PI);
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < Nt; ++i) {
        double ph = 0.0, g[3] = {0, 0, 0};
        for (int64_t j = 0; j < Ns; ++j) {
            const double dx = tpos[3 * i] - spos[3 * j], dy = tpos[3 * i + 1] - spos[3 * j + 1], dz = tpos[3 * i + 2] - spos[3 * j + 2];
            if (coincident(rule, dx, dy, dz)) continue;
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double r = std::sqrt(r2);
            ph += q[j] / r;
            const double f = q[j] / (r2 * r);
            g[0] -= f * dx; g[1] -= f * dy; g[2] -= f * dz;
        }
        if (pot) pot[i] = -ph * inv4pi;
        if (field) for (int c = 0; c < 3; ++c) field[3 * i + c] = g[c] * inv4pi;
    }
}
// number of OpenMP threads used by the following calls (bench.py's one-thread cpu_baseline leg); n < 1 restores the default
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    omp_set_num_threads(n >= 1 ? n : omp_get_num_procs());
#else
    (void)n;
#endif
}
int orc_num_threads() {
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp single
        n = omp_get_num_threads();
    }
#endif
    return n;
}

}  // extern "C"
