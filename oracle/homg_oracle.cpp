// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
//
// Plain, slow, single-threaded C++ restatement of the high-occupancy multigrid
// (HOMG) cycle of arxiv 1108.2045, written from PAPER.md alone.  It shares no
// code with the CUDA path (paper_1108_2045_b200/csrc) and neither imports the
// other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may build, load or call this file.
//
// What is here (PAPER.md line numbers; DESIGN.md lists every reading R1..):
//   apply_A / residual       A = -div(k grad) on a 5-/7-point stencil, Dirichlet u=0
//                            (Eq.1, L89-93 Eq.4; sign: DESIGN.md R1)
//   jacobi                   damped Jacobi, Eq. 3: v <- v + w_p ((sum_nb v - 2d v) + h^2 g)   (L53-67 Eq.2-3)
//   restrict_fw              weighted-average restriction P, nested (L47, L67, L73)
//   prolong                  linear (bi-/tri-linear) interpolation S     (L47, L51)
//   homg  alg=0 "L"          the literal single-array HOMG iteration: every whole-grid
//                            iteration relaxes the level-m lattice and interpolates the
//                            previous-iteration variations everywhere else (L51, L69, L113),
//                            MFMG schedule (L69-71), residual restart (L75)
//   homg  alg=1 "H"          the same cycle carried on per-level arrays (what the GPU
//                            implements); must equal L to rounding
//   vcycle                   classic V(eta1,eta2) (L47)
//   homg_p2                  section 3 (L77-85): the literal iteration on a 2-D grid of 2^k nodes per side
//   dense_solve / assemble   dense LU of A u = f on tiny grids (fixed point of the cycle)
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): dense LU fixed point, Laplacian
// eigenvectors with closed-form Jacobi factors, restriction/prolongation mode
// formulas and adjointness, the L113 spike/pyramid closed forms, L == H, linearity,
// O(h^2) against manufactured solutions, the paper's printed L1 errors (L119, loose),
// linear cost.  Parity unpinned: the "31 iterations" count of L113 (no reading of the
// missing Fig. 1 reproduces an odd total; R3).
//
// Arithmetic is carried in the template scalar T (double, or float for the fp32
// configs); norms are always accumulated in double.  Arrays are dense, C order,
// dims = nodes per axis including the Dirichlet boundary, dims[0] slowest.
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>

namespace {

unsigned long long g_relax_updates = 0;   // Jacobi node updates (cost pin)
unsigned long long g_move_updates = 0;    // node updates in interpolation / injection moves

struct Grid {
    int nd;            // 2 or 3
    int64_t n[3];      // n[0]=nz (1 when nd==2), n[1]=ny, n[2]=nx
    int64_t st[3];     // element strides
    int a0() const { return 3 - nd; }
    int64_t size() const { return n[0] * n[1] * n[2]; }
    int64_t idx(const int64_t p[3]) const { return p[0] * st[0] + p[1] * st[1] + p[2] * st[2]; }
    bool on_boundary(const int64_t p[3]) const {
        for (int a = a0(); a < 3; ++a)
            if (p[a] == 0 || p[a] == n[a] - 1) return true;
        return false;
    }
};

Grid make_grid(int nd, const int64_t* dims) {
    Grid G;
    G.nd = nd;
    G.n[0] = 1; G.n[1] = 1; G.n[2] = 1;
    for (int a = 0; a < nd; ++a) G.n[3 - nd + a] = dims[a];
    G.st[2] = 1; G.st[1] = G.n[2]; G.st[0] = G.n[1] * G.n[2];
    return G;
}

Grid coarser(const Grid& F) {
    int64_t d[3];
    for (int a = 0; a < F.nd; ++a) d[a] = (F.n[F.a0() + a] - 1) / 2 + 1;
    return make_grid(F.nd, d);
}

Grid finer(const Grid& C) {
    int64_t d[3];
    for (int a = 0; a < C.nd; ++a) d[a] = 2 * (C.n[C.a0() + a] - 1) + 1;
    return make_grid(C.nd, d);
}

#define FOR_NODES(G, p)                                     \
    for (int64_t p##0 = 0; p##0 < (G).n[0]; ++p##0)         \
        for (int64_t p##1 = 0; p##1 < (G).n[1]; ++p##1)     \
            for (int64_t p##2 = 0; p##2 < (G).n[2]; ++p##2)

// ---------------------------------------------------------------------------
// The operator at one node.  `v` and `kc` are addressed with element strides
// `st[]` (so the same code serves a per-level array, st = the array's strides,
// and the literal single-array algorithm, st = 2^m times the fine strides:
// PAPER.md L65 Eq.3, "l = 2^m").  ih2 = 1/h_m^2.
//   constant coefficient: (A v)(p) = (2d v(p) - sum_nb v) / h^2
//   nodal coefficient k : (A v)(p) = sum_faces kf (v(p) - v(q)) / h^2,
//                         kf = 2 k_p k_q / (k_p + k_q)   (R11)
// ---------------------------------------------------------------------------
template <class T>
inline T opA_node(int nd, const T* v, const T* kc, int64_t c, const int64_t st[3], T ih2) {
    if (!kc) {
        T s = 0;
        for (int a = 3 - nd; a < 3; ++a) s += v[c - st[a]] + v[c + st[a]];
        return (T(2 * nd) * v[c] - s) * ih2;
    }
    T acc = 0;
    for (int a = 3 - nd; a < 3; ++a) {
        for (int sg = -1; sg <= 1; sg += 2) {
            int64_t q = c + sg * st[a];
            T kf = T(2) * kc[c] * kc[q] / (kc[c] + kc[q]);
            acc += kf * (v[c] - v[q]);
        }
    }
    return acc * ih2;
}

template <class T>
inline T diag_node(int nd, const T* kc, int64_t c, const int64_t st[3], T ih2) {
    if (!kc) return T(2 * nd) * ih2;
    T acc = 0;
    for (int a = 3 - nd; a < 3; ++a) {
        for (int sg = -1; sg <= 1; sg += 2) {
            int64_t q = c + sg * st[a];
            acc += T(2) * kc[c] * kc[q] / (kc[c] + kc[q]);
        }
    }
    return acc * ih2;
}

// damped Jacobi at one node.
//   constant coefficient: Eq. 3 (L65) as printed, in the sign convention of DESIGN.md R1 (A = -lap,
//   g = the paper's -P_m f):   v + w_p ((sum_nb v - 2d v) + h_l^2 g),   w_p = w / 2d,  h2 = h_l^2.
//   The three multiply-adds are single fused operations (std::fma), in Eq. 3's order: neighbour sum
//   minus 2d v, plus h^2 g, times w_p, added to v (R14; the GPU uses FMA in the same places).
//   nodal coefficient k: no equation in the paper; v + w (g - A v) / D with the flux-form A, D (R11).
template <class T>
inline T jacobi_node(int nd, const T* v, const T* kc, int64_t c, const int64_t st[3], T ih2, T w, T g, T h2, T wp) {
    if (!kc) {
        T s = 0;
        for (int a = 3 - nd; a < 3; ++a) s += v[c - st[a]] + v[c + st[a]];
        T t = std::fma(-T(2 * nd), v[c], s);
        t = std::fma(h2, g, t);
        return std::fma(wp, t, v[c]);
    }
    T Av = opA_node(nd, v, kc, c, st, ih2);
    T D = diag_node(nd, kc, c, st, ih2);
    return v[c] + w * (g - Av) / D;
}

template <class T>
void apply_A(const Grid& G, double h, const T* kc, const T* v, T* out) {
    T ih2 = T(1.0 / (h * h));
    FOR_NODES(G, p) {
        int64_t p[3] = {p0, p1, p2};
        int64_t c = G.idx(p);
        out[c] = G.on_boundary(p) ? T(0) : opA_node(G.nd, v, kc, c, G.st, ih2);
    }
}

// r = f - A u on interior nodes, 0 on the boundary; returns sum r^2 in double
template <class T>
double residual(const Grid& G, double h, const T* kc, const T* u, const T* f, T* r) {
    T ih2 = T(1.0 / (h * h));
    double s2 = 0;
    FOR_NODES(G, p) {
        int64_t p[3] = {p0, p1, p2};
        int64_t c = G.idx(p);
        T rv = 0;
        if (!G.on_boundary(p)) rv = f[c] - opA_node(G.nd, u, kc, c, G.st, ih2);
        if (r) r[c] = rv;
        s2 += double(rv) * double(rv);
    }
    return s2;
}

template <class T>
void jacobi(const Grid& G, double h, const T* kc, double omega, const T* v, const T* g, T* out) {
    T ih2 = T(1.0 / (h * h));
    T w = T(omega);
    T h2 = T(h * h), wp = T(omega / double(2 * G.nd));
    FOR_NODES(G, p) {
        int64_t p[3] = {p0, p1, p2};
        int64_t c = G.idx(p);
        if (G.on_boundary(p)) { out[c] = 0; continue; }
        out[c] = jacobi_node(G.nd, v, kc, c, G.st, ih2, w, g[c], h2, wp);
        ++g_relax_updates;
    }
}

// Full weighting: coarse interior node I gets sum_{delta in {-1,0,1}^d}
// 2^(-d-|delta|_1) fine(2I+delta); coarse boundary entries are 0.
template <class T>
void restrict_fw(const Grid& F, const T* in, T* out) {
    Grid C = coarser(F);
    int nd = F.nd, a0 = F.a0();
    FOR_NODES(C, P) {
        int64_t P[3] = {P0, P1, P2};
        int64_t cidx = C.idx(P);
        if (C.on_boundary(P)) { out[cidx] = 0; continue; }
        T acc = 0;
        int64_t lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
        for (int a = a0; a < 3; ++a) { lo[a] = -1; hi[a] = 1; }
        for (int64_t d0 = lo[0]; d0 <= hi[0]; ++d0)
            for (int64_t d1 = lo[1]; d1 <= hi[1]; ++d1)
                for (int64_t d2 = lo[2]; d2 <= hi[2]; ++d2) {
                    int64_t q[3] = {2 * P[0] + d0, 2 * P[1] + d1, 2 * P[2] + d2};
                    int m1 = int(std::llabs(d0) + std::llabs(d1) + std::llabs(d2));
                    T wgt = T(1.0 / double(1 << (nd + m1)));
                    acc += wgt * in[F.idx(q)];
                }
        out[cidx] = acc;
        ++g_move_updates;
    }
}

// Multilinear interpolation of a lattice of spacing `s` (in units of the target
// grid) onto every node of the target grid T: value at p = sum over the 2^d
// corners of the enclosing cell of prod_a (1 - t_a/s | t_a/s) * src(corner).
// `src` is addressed by (corner index) * sst[a].  s = 2: one-level prolongation.
template <class T>
inline T interp_node(int nd, const int64_t p[3], int64_t s, const T* src, const int64_t sst[3]) {
    int a0 = 3 - nd;
    int64_t base[3] = {0, 0, 0};
    T wl[3] = {1, 1, 1}, wh[3] = {0, 0, 0};
    for (int a = a0; a < 3; ++a) {
        base[a] = p[a] / s;
        int64_t t = p[a] - base[a] * s;
        wh[a] = T(double(t) / double(s));
        wl[a] = T(1) - wh[a];
    }
    T acc = 0;
    for (int c0 = 0; c0 <= (a0 <= 0); ++c0)
        for (int c1 = 0; c1 <= (a0 <= 1); ++c1)
            for (int c2 = 0; c2 <= 1; ++c2) {
                int cc[3] = {c0, c1, c2};
                T w = 1;
                bool zero = false;
                for (int a = a0; a < 3; ++a) {
                    T wa = cc[a] ? wh[a] : wl[a];
                    if (wa == T(0)) zero = true;
                    w *= wa;
                }
                if (zero) continue;   // also keeps corners past the last node from being read
                int64_t q = 0;
                for (int a = a0; a < 3; ++a) q += (base[a] + cc[a]) * sst[a];
                acc += w * src[q];
            }
    return acc;
}

// one-level prolongation S^ : coarse per-level array -> fine per-level array
template <class T>
void prolong(const Grid& C, const T* in, T* out) {
    Grid F = finer(C);
    FOR_NODES(F, p) {
        int64_t p[3] = {p0, p1, p2};
        out[F.idx(p)] = interp_node(F.nd, p, 2, in, C.st);
        ++g_move_updates;
    }
}

// ---------------------------------------------------------------------------
// Hierarchy description shared by L, H and V.
// ---------------------------------------------------------------------------
template <class T>
struct Hier {
    int levels;
    std::vector<Grid> G;            // G[0] finest
    std::vector<double> h;          // h[m] = 2^m h
    std::vector<std::vector<T>> k;  // nodal coefficient sampled on every level (empty: constant)
    const T* kptr(int m) const { return k.empty() ? nullptr : k[m].data(); }
};

template <class T>
bool build_hier(Hier<T>& H, int nd, const int64_t* dims, int levels, double h, const T* kc) {
    if (nd < 2 || nd > 3 || levels < 1) return false;
    for (int a = 0; a < nd; ++a) {
        int64_t q = int64_t(1) << (levels - 1);
        if (dims[a] < 3 || (dims[a] - 1) % q != 0 || (dims[a] - 1) / q < 2) return false;
    }
    H.levels = levels;
    H.G.clear(); H.h.clear(); H.k.clear();
    H.G.push_back(make_grid(nd, dims));
    H.h.push_back(h);
    for (int m = 1; m < levels; ++m) {
        H.G.push_back(coarser(H.G[m - 1]));
        H.h.push_back(2 * H.h[m - 1]);
    }
    if (kc) {
        // level-m coefficient = k sampled at the level-m lattice nodes (R11)
        H.k.resize(levels);
        H.k[0].assign(kc, kc + H.G[0].size());
        for (int m = 1; m < levels; ++m) {
            const Grid& C = H.G[m];
            const Grid& F = H.G[m - 1];
            H.k[m].resize(C.size());
            FOR_NODES(C, P) {
                int64_t P[3] = {P0, P1, P2};
                int64_t q[3] = {2 * P0, 2 * P1, 2 * P2};
                H.k[m][C.idx(P)] = H.k[m - 1][F.idx(q)];
            }
        }
    }
    return true;
}

// restricted sources g_0 = r, g_m = P g_{m-1}   ("nested partial reductions")
template <class T>
void restrict_chain(const Hier<T>& H, std::vector<std::vector<T>>& g) {
    for (int m = 1; m < H.levels; ++m) {
        g[m].assign(H.G[m].size(), T(0));
        restrict_fw(H.G[m - 1], g[m - 1].data(), g[m].data());
    }
}

// ---------------------------------------------------------------------------
// Algorithm L — the literal HOMG iteration on ONE fine-grid array.
// One whole-grid iteration at level m:
//   lattice nodes (every index a multiple of l=2^m) relax with the stride-l stencil
//   (Eq.3), boundary lattice nodes stay 0; every other node adds the multilinear
//   interpolation of the lattice nodes' previous-iteration variation cur-prev
//   ("interpolations of the previous iteration variations"; one-iteration delay, L113).
// ---------------------------------------------------------------------------
template <class T>
void iteration_L(const Hier<T>& H, int m, double omega, const std::vector<T>& gm,
                 std::vector<T>& cur, std::vector<T>& prev, std::vector<T>& nxt, std::vector<T>& var) {
    const Grid& F = H.G[0];
    const Grid& Gm = H.G[m];
    int nd = F.nd, a0 = F.a0();
    int64_t l = int64_t(1) << m;
    int64_t stl[3] = {F.st[0] * l, F.st[1] * l, F.st[2] * l};
    T ih2 = T(1.0 / (H.h[m] * H.h[m]));
    T w = T(omega);
    T h2 = T(H.h[m] * H.h[m]), wp = T(omega / double(2 * nd));
    const T* kc = H.kptr(0);
    // variation of every node in the previous iteration
    for (int64_t i = 0; i < F.size(); ++i) var[i] = cur[i] - prev[i];
    FOR_NODES(F, p) {
        int64_t p[3] = {p0, p1, p2};
        int64_t c = F.idx(p);
        bool lattice = true;
        for (int a = a0; a < 3; ++a) lattice = lattice && (p[a] % l == 0);
        if (lattice) {
            if (F.on_boundary(p)) { nxt[c] = 0; continue; }
            int64_t P[3] = {p[0] / l, p[1] / l, p[2] / l};
            nxt[c] = jacobi_node(nd, cur.data(), kc, c, stl, ih2, w, gm[Gm.idx(P)], h2, wp);
            ++g_relax_updates;
        } else {
            nxt[c] = cur[c] + interp_node(nd, p, l, var.data(), stl);
            ++g_move_updates;
        }
    }
    prev.swap(cur);
    cur.swap(nxt);
}

template <class T>
double cycle_L(const Hier<T>& H, double omega, const int* slv, const int* sit, int slen,
               const T* f, T* u, long max_iters, T* cur_out) {
    const Grid& F = H.G[0];
    std::vector<std::vector<T>> g(H.levels);
    g[0].assign(F.size(), T(0));
    double n2 = residual(F, H.h[0], H.kptr(0), u, f, g[0].data());
    restrict_chain(H, g);
    std::vector<T> cur(F.size(), T(0)), prev(F.size(), T(0)), nxt(F.size(), T(0)), var(F.size(), T(0));
    long done = 0;
    for (int s = 0; s < slen && (max_iters < 0 || done < max_iters); ++s)
        for (int it = 0; it < sit[s] && (max_iters < 0 || done < max_iters); ++it, ++done)
            iteration_L(H, slv[s], omega, g[slv[s]], cur, prev, nxt, var);
    if (cur_out) std::memcpy(cur_out, cur.data(), sizeof(T) * F.size());
    for (int64_t i = 0; i < F.size(); ++i) u[i] += cur[i];
    return std::sqrt(n2);
}

// ---------------------------------------------------------------------------
// Algorithm H — the same cycle on per-level arrays.
//   e[m]  : values of the correction on the level-m lattice (current when at level m)
//   a[m]  : increments the level-m lattice owes to all finer nodes, not yet delivered
//   dl,dp : last and last-but-one Jacobi increments of the latest visit
// ---------------------------------------------------------------------------
template <class T>
double cycle_H(const Hier<T>& H, double omega, const int* slv, const int* sit, int slen,
               const T* f, T* u) {
    int L = H.levels;
    std::vector<std::vector<T>> g(L), e(L), a(L);
    g[0].assign(H.G[0].size(), T(0));
    double n2 = residual(H.G[0], H.h[0], H.kptr(0), u, f, g[0].data());
    restrict_chain(H, g);
    for (int m = 0; m < L; ++m) { e[m].assign(H.G[m].size(), T(0)); a[m].assign(H.G[m].size(), T(0)); }

    int cur = -1;                  // current level, -1 before the first visit
    std::vector<T> dl, dp;         // on level `cur`
    for (int s = 0; s < slen; ++s) {
        int t = slv[s], eta = sit[s];
        const Grid& Gt = H.G[t];
        std::vector<T> d0(Gt.size(), T(0));
        if (cur >= 0) {
            // ---- move ----
            if (t < cur) {
                for (int m = cur; m > t; --m) {           // deliver level m -> m-1
                    const Grid& Fm = H.G[m - 1];
                    std::vector<T> inc(Fm.size());
                    prolong(H.G[m], a[m].data(), inc.data());
                    FOR_NODES(Fm, p) {
                        int64_t p[3] = {p0, p1, p2};
                        int64_t c = Fm.idx(p);
                        bool coin = true;
                        for (int ax = Fm.a0(); ax < 3; ++ax) coin = coin && (p[ax] % 2 == 0);
                        if (coin) {
                            int64_t P[3] = {p[0] / 2, p[1] / 2, p[2] / 2};
                            e[m - 1][c] = e[m][H.G[m].idx(P)];
                        } else {
                            e[m - 1][c] += inc[c];
                        }
                        if (m - 1 >= 1) a[m - 1][c] += inc[c];
                    }
                    std::fill(a[m].begin(), a[m].end(), T(0));
                }
            } else if (t > cur) {
                for (int m = cur + 1; m <= t; ++m) {      // inject level m-1 -> m
                    const Grid& C = H.G[m];
                    const Grid& Fm = H.G[m - 1];
                    FOR_NODES(C, P) {
                        int64_t P[3] = {P0, P1, P2};
                        int64_t q[3] = {2 * P0, 2 * P1, 2 * P2};
                        e[m][C.idx(P)] = e[m - 1][Fm.idx(q)];
                        ++g_move_updates;
                    }
                }
            }
            // ---- carried variation d0: what every level-t lattice node did in the
            //      iteration just before this visit ----
            if (t >= cur) {
                int64_t s2 = int64_t(1) << (t - cur);
                const Grid& V = H.G[cur];
                FOR_NODES(Gt, P) {
                    int64_t P[3] = {P0, P1, P2};
                    int64_t q[3] = {P0 * s2, P1 * s2, P2 * s2};
                    d0[Gt.idx(P)] = dl[V.idx(q)];
                }
            } else {
                std::vector<T> tmp = dp;
                for (int m = cur; m > t; --m) {
                    std::vector<T> fine(H.G[m - 1].size());
                    prolong(H.G[m], tmp.data(), fine.data());
                    tmp.swap(fine);
                }
                int64_t s2 = int64_t(1) << (cur - t);
                const Grid& V = H.G[cur];
                FOR_NODES(Gt, p) {
                    int64_t p[3] = {p0, p1, p2};
                    bool coin = true;
                    for (int ax = Gt.a0(); ax < 3; ++ax) coin = coin && (p[ax] % s2 == 0);
                    int64_t c = Gt.idx(p);
                    if (coin) {
                        int64_t P[3] = {p[0] / s2, p[1] / s2, p[2] / s2};
                        d0[c] = dl[V.idx(P)];
                    } else {
                        d0[c] = tmp[c];
                    }
                }
            }
        }
        // ---- eta Jacobi sweeps on level t ----
        std::vector<T> v0 = e[t];              // v^0
        std::vector<T> vk = e[t], vkm1, vkm2;  // v^k, v^{k-1}, v^{k-2}
        for (int it = 0; it < eta; ++it) {
            vkm2.swap(vkm1);
            vkm1.swap(vk);
            vk.assign(Gt.size(), T(0));
            jacobi(Gt, H.h[t], H.kptr(t), omega, vkm1.data(), g[t].data(), vk.data());
        }
        // now vk = v^eta, vkm1 = v^{eta-1}, vkm2 = v^{eta-2} (when eta >= 2)
        dl.assign(Gt.size(), T(0));
        std::vector<T> ndp(Gt.size(), T(0));
        for (int64_t i = 0; i < Gt.size(); ++i) {
            T D = (d0[i] + vkm1[i]) - v0[i];             // variations interpolated during the visit
            if (t >= 1) a[t][i] += D;
            dl[i] = vk[i] - vkm1[i];
            ndp[i] = (eta >= 2) ? (vkm1[i] - vkm2[i]) : d0[i];
        }
        dp.swap(ndp);
        e[t] = vk;
        cur = t;
    }
    const Grid& F = H.G[0];
    for (int64_t i = 0; i < F.size(); ++i) u[i] += e[0][i];
    return std::sqrt(n2);
}

// ---------------------------------------------------------------------------
// Dense LU with partial pivoting (double).  Unknowns = interior nodes, C order.
// ---------------------------------------------------------------------------
bool lu_solve(std::vector<double>& A, std::vector<double>& b, int64_t N) {
    for (int64_t c = 0; c < N; ++c) {
        int64_t piv = c;
        for (int64_t r = c + 1; r < N; ++r)
            if (std::fabs(A[r * N + c]) > std::fabs(A[piv * N + c])) piv = r;
        if (A[piv * N + c] == 0.0) return false;
        if (piv != c) {
            for (int64_t j = 0; j < N; ++j) std::swap(A[c * N + j], A[piv * N + j]);
            std::swap(b[c], b[piv]);
        }
        for (int64_t r = c + 1; r < N; ++r) {
            double fct = A[r * N + c] / A[c * N + c];
            if (fct == 0.0) continue;
            for (int64_t j = c; j < N; ++j) A[r * N + j] -= fct * A[c * N + j];
            b[r] -= fct * b[c];
        }
    }
    for (int64_t r = N - 1; r >= 0; --r) {
        double s = b[r];
        for (int64_t j = r + 1; j < N; ++j) s -= A[r * N + j] * b[j];
        b[r] = s / A[r * N + r];
    }
    return true;
}

// interior numbering
int64_t interior_count(const Grid& G) {
    int64_t N = 1;
    for (int a = G.a0(); a < 3; ++a) N *= (G.n[a] - 2);
    return N;
}

void interior_index(const Grid& G, std::vector<int64_t>& map) {
    map.assign(G.size(), -1);
    int64_t cnt = 0;
    FOR_NODES(G, p) {
        int64_t p[3] = {p0, p1, p2};
        if (!G.on_boundary(p)) map[G.idx(p)] = cnt++;
    }
}

// dense matrix of A on the interior unknowns, built column by column from apply_A
template <class T>
void assemble(const Grid& G, double h, const T* kc, std::vector<double>& A) {
    int64_t N = interior_count(G);
    std::vector<int64_t> map;
    interior_index(G, map);
    A.assign(N * N, 0.0);
    std::vector<T> v(G.size(), T(0)), out(G.size());
    for (int64_t c = 0; c < G.size(); ++c) {
        if (map[c] < 0) continue;
        v[c] = 1;
        apply_A(G, h, kc, v.data(), out.data());
        v[c] = 0;
        for (int64_t r = 0; r < G.size(); ++r)
            if (map[r] >= 0) A[map[r] * N + map[c]] = double(out[r]);
    }
}

template <class T>
bool dense_solve(const Grid& G, double h, const T* kc, const T* f, T* u) {
    int64_t N = interior_count(G);
    std::vector<int64_t> map;
    interior_index(G, map);
    std::vector<double> A, b(N);
    assemble(G, h, kc, A);
    for (int64_t c = 0; c < G.size(); ++c)
        if (map[c] >= 0) b[map[c]] = double(f[c]);
    if (!lu_solve(A, b, N)) return false;
    for (int64_t c = 0; c < G.size(); ++c) u[c] = map[c] >= 0 ? T(b[map[c]]) : T(0);
    return true;
}

// ---------------------------------------------------------------------------
// Classic V(eta1, eta2)
// ---------------------------------------------------------------------------
template <class T>
void vcycle_rec(const Hier<T>& H, int m, double omega, int eta1, int eta2, std::vector<T>& v,
                const std::vector<T>& g) {
    const Grid& G = H.G[m];
    if (m == H.levels - 1) {     // (c) solve the coarsest residual equation exactly
        dense_solve(G, H.h[m], H.kptr(m), g.data(), v.data());
        return;
    }
    std::vector<T> tmp(G.size());
    for (int it = 0; it < eta1; ++it) {          // (a)
        jacobi(G, H.h[m], H.kptr(m), omega, v.data(), g.data(), tmp.data());
        v.swap(tmp);
    }
    std::vector<T> r(G.size()), gc(H.G[m + 1].size()), ec(H.G[m + 1].size(), T(0));
    residual(G, H.h[m], H.kptr(m), v.data(), g.data(), r.data());
    restrict_fw(G, r.data(), gc.data());         // (b)
    vcycle_rec(H, m + 1, omega, eta1, eta2, ec, gc);
    prolong(H.G[m + 1], ec.data(), tmp.data());  // (d)
    for (int64_t i = 0; i < G.size(); ++i) v[i] += tmp[i];
    for (int it = 0; it < eta2; ++it) {          // (e)
        jacobi(G, H.h[m], H.kptr(m), omega, v.data(), g.data(), tmp.data());
        v.swap(tmp);
    }
}

// ---------------------------------------------------------------------------
// MFMG schedule (Fig. 1 is missing from PAPER.md — DESIGN.md R3).
//   its(m) = min(2^(M-m+1), MaxI): 2 on the coarsest level, doubling per finer level.
//   kind 0 "C": M, then for k=M-1..0: k, and if k>0: k+1
//   kind 1 "A": M, M-1, then for k=M-2..0: k+2, k+1, k
//   kind 2 sawtooth: for k=M..0: M, M-1, .., k
// ---------------------------------------------------------------------------
int make_schedule(int kind, int levels, int maxI, int* lv, int* it, int cap) {
    if (levels < 1 || maxI < 1) return -1;
    int M = levels - 1;
    std::vector<int> seq;
    if (kind == 0) {
        seq.push_back(M);
        for (int k = M - 1; k >= 0; --k) { seq.push_back(k); if (k > 0) seq.push_back(k + 1); }
    } else if (kind == 1) {
        seq.push_back(M);
        if (M >= 1) seq.push_back(M - 1);
        for (int k = M - 2; k >= 0; --k) { seq.push_back(k + 2); seq.push_back(k + 1); seq.push_back(k); }
    } else if (kind == 2) {
        for (int k = M; k >= 0; --k)
            for (int j = M; j >= k; --j) seq.push_back(j);
    } else {
        return -1;
    }
    if (int(seq.size()) > cap) return -int(seq.size());
    for (size_t i = 0; i < seq.size(); ++i) {
        lv[i] = seq[i];
        long its = 1L << std::min(M - seq[i] + 1, 30);
        it[i] = int(std::min<long>(its, maxI));
    }
    return int(seq.size());
}

template <class T>
int run_homg(int alg, int nd, const int64_t* dims, int levels, double h, const void* kc, double omega,
             const int* slv, const int* sit, int slen, const void* f, void* u, int ncycles,
             void* u_hist, double* norms) {
    Hier<T> H;
    if (!build_hier<T>(H, nd, dims, levels, h, static_cast<const T*>(kc))) return 1;
    if (slen < 1 || slv[slen - 1] != 0) return 2;
    for (int s = 0; s < slen; ++s)
        if (slv[s] < 0 || slv[s] >= levels || sit[s] < 1) return 2;
    T* uu = static_cast<T*>(u);
    const T* ff = static_cast<const T*>(f);
    int64_t N = H.G[0].size();
    for (int c = 0; c < ncycles; ++c) {
        double nr = alg == 0 ? cycle_L(H, omega, slv, sit, slen, ff, uu, -1, (T*)nullptr)
                             : cycle_H(H, omega, slv, sit, slen, ff, uu);
        if (norms) norms[c] = nr;
        if (u_hist) std::memcpy(static_cast<T*>(u_hist) + int64_t(c) * N, uu, sizeof(T) * N);
    }
    if (norms) norms[ncycles] = std::sqrt(residual(H.G[0], h, H.kptr(0), uu, ff, (T*)nullptr));
    return 0;
}

template <class T>
int run_vcycle(int nd, const int64_t* dims, int levels, double h, const void* kc, double omega, int eta1,
               int eta2, const void* f, void* u, int ncycles, void* u_hist, double* norms) {
    Hier<T> H;
    if (!build_hier<T>(H, nd, dims, levels, h, static_cast<const T*>(kc))) return 1;
    T* uu = static_cast<T*>(u);
    const T* ff = static_cast<const T*>(f);
    int64_t N = H.G[0].size();
    std::vector<T> v(uu, uu + N), g(ff, ff + N);
    for (int c = 0; c < ncycles; ++c) {
        if (norms) norms[c] = std::sqrt(residual(H.G[0], h, H.kptr(0), v.data(), ff, (T*)nullptr));
        vcycle_rec(H, 0, omega, eta1, eta2, v, g);
        if (u_hist) std::memcpy(static_cast<T*>(u_hist) + int64_t(c) * N, v.data(), sizeof(T) * N);
    }
    if (norms) norms[ncycles] = std::sqrt(residual(H.G[0], h, H.kptr(0), v.data(), ff, (T*)nullptr));
    std::memcpy(uu, v.data(), sizeof(T) * N);
    return 0;
}

// ---------------------------------------------------------------------------
// Mixed-precision outer loop.  PAPER.md L75: "the residual equation is used to restart
// the cycles" — the restart is a defect-correction loop, so the correction cycle may run in a lower
// precision than the residual:  u, f and r = f - A u in fp64;  r rounded to fp32;  ONE HOMG cycle in fp32
// on A e = r from e = 0 (Algorithm H, coefficient k rounded to fp32);  u += e in fp64.
// ---------------------------------------------------------------------------
int run_homg_mixed(int nd, const int64_t* dims, int levels, double h, const double* kc, double omega,
                   const int* slv, const int* sit, int slen, const double* f, double* u, int ncycles,
                   double* u_hist, double* norms) {
    Hier<double> Hd;
    if (!build_hier<double>(Hd, nd, dims, levels, h, kc)) return 1;
    const Grid& F = Hd.G[0];
    const int64_t N = F.size();
    std::vector<float> k32;
    if (kc) { k32.resize(N); for (int64_t i = 0; i < N; ++i) k32[i] = float(kc[i]); }
    Hier<float> Hf;
    if (!build_hier<float>(Hf, nd, dims, levels, h, kc ? k32.data() : nullptr)) return 1;
    std::vector<double> r(N);
    std::vector<float> r32(N), e32(N);
    for (int c = 0; c < ncycles; ++c) {
        double n2 = residual(F, h, Hd.kptr(0), u, f, r.data());
        if (norms) norms[c] = std::sqrt(n2);
        for (int64_t i = 0; i < N; ++i) { r32[i] = float(r[i]); e32[i] = 0.0f; }
        cycle_H<float>(Hf, omega, slv, sit, slen, r32.data(), e32.data());
        for (int64_t i = 0; i < N; ++i) u[i] += double(e32[i]);
        if (u_hist) std::memcpy(u_hist + int64_t(c) * N, u, sizeof(double) * N);
    }
    if (norms) norms[ncycles] = std::sqrt(residual(F, h, Hd.kptr(0), u, f, (double*)nullptr));
    return 0;
}


// ---------------------------------------------------------------------------
// Algorithm P — PAPER.md section 3 (L77-85), "Power of two size grids": the literal HOMG iteration on a 2-D grid
// with N = 2^k nodes per side (N-1 intervals: not nestable).  Fig. 2 is not in the file; the reading is DESIGN.md R19:
//   * the grid is divided into four subdomains of N/2 x N/2 nodes (L79, L83: "four subdomains with a power of two
//     nodes per side"); per axis a node belongs to the LOW half (index < N/2) or the HIGH half;
//   * the level-m coarse points of a subdomain are marked "relative to the corresponding external corner" (L83): per
//     axis the low half's lattice is {i l}, the high half's {N-1 - i l}, l = 2^m, i = 0 .. N/(2l).  The last point,
//     i = N/(2l), lies "just outside the corresponding subdomain" (L85) — the central points without which "some coarse
//     modes, like the zero mode, can not be resolved" (`central` = 0 leaves them out: the pin that shows exactly that);
//   * "We perform relaxations in all the marked points and interpolations on the rest of the fine grid" (L85): a marked
//     interior node relaxes with the stride-l stencil of Eq. 3 IN THE FINE ARRAY (its neighbours at distance l need not be
//     marked; an index outside the grid counts as the Dirichlet value 0); its source is the weighted-average restriction
//     P_m r on ITS lattice: each of the 2 x 2 anchor combinations is a nested lattice of the (N+1)-node grid obtained by
//     adding one ghost row / column (value 0) beyond the side opposite to the anchor, so "nested partial reductions"
//     (L73) apply to each unchanged;
//   * every other node adds the bilinear interpolation of the previous-iteration variations of the marked nodes of ITS
//     OWN subdomain's lattice: "The interpolations make use only of points in the same subdomain" (L85).
// Everything else (schedule, restart, one-iteration delay, Eq. 3 arithmetic) is Algorithm L's.
// ---------------------------------------------------------------------------
struct P2Lattice {
    int64_t N, l;
    bool central;
    int64_t last() const { return central ? N / 2 : N / 2 - 1; }      // largest distance from the anchor that is marked
    // is coordinate x on the low- / high-anchored lattice?  *anchor = 0 (low) or 1 (high); level 0: every x, anchor 0
    bool on(int64_t x, int* anchor) const {
        if (x % l == 0 && x <= last()) { *anchor = 0; return true; }
        const int64_t t = N - 1 - x;
        if (t % l == 0 && t <= last()) { *anchor = 1; return true; }
        return false;
    }
};

// E[ay][ax][m]: nested full weighting of the residual on the lattice anchored at corner (ay, ax); arrays of
// (N / 2^m + 1)^2 entries indexed FROM THE ANCHOR, the last row / column being the ghost (0)
template <class T>
void p2_restrict_all(int64_t N, int levels, const T* r, std::vector<std::vector<T>> E[2][2]) {
    for (int ay = 0; ay < 2; ++ay)
        for (int ax = 0; ax < 2; ++ax) {
            auto& H = E[ay][ax];
            H.assign(levels, std::vector<T>());
            H[0].assign(size_t((N + 1) * (N + 1)), T(0));
            for (int64_t i = 0; i < N; ++i)
                for (int64_t j = 0; j < N; ++j)
                    H[0][size_t(i * (N + 1) + j)] = r[(ay ? N - 1 - i : i) * N + (ax ? N - 1 - j : j)];
            int64_t n = N + 1;
            for (int m = 1; m < levels; ++m) {
                int64_t d[2] = {n, n};
                Grid F = make_grid(2, d);
                n = (n - 1) / 2 + 1;
                H[m].assign(size_t(n * n), T(0));
                restrict_fw(F, H[m - 1].data(), H[m].data());
            }
        }
}

template <class T>
void iteration_P(int64_t N, int m, double h, double omega, bool central, std::vector<std::vector<T>> E[2][2],
                 std::vector<T>& cur, std::vector<T>& prev, std::vector<T>& nxt, std::vector<T>& var) {
    const int64_t l = int64_t(1) << m;
    const P2Lattice Lt{N, l, central};
    const double hm = double(l) * h;
    const T h2 = T(hm * hm), wp = T(omega / 4.0);
    for (int64_t i = 0; i < N * N; ++i) var[size_t(i)] = cur[size_t(i)] - prev[size_t(i)];
    auto at = [&](int64_t y, int64_t x) -> T { return (y < 0 || y >= N || x < 0 || x >= N) ? T(0) : cur[size_t(y * N + x)]; };
    for (int64_t y = 0; y < N; ++y)
        for (int64_t x = 0; x < N; ++x) {
            const size_t c = size_t(y * N + x);
            if (y == 0 || y == N - 1 || x == 0 || x == N - 1) { nxt[c] = 0; continue; }
            int ay = 0, ax = 0;
            if (Lt.on(y, &ay) && Lt.on(x, &ax)) {
                // relaxation, Eq. 3 (same three fused multiply-adds as jacobi_node)
                const int64_t nl = N / l + 1;
                const int64_t iy = (ay ? N - 1 - y : y) / l, ix = (ax ? N - 1 - x : x) / l;
                const T g = E[ay][ax][m][size_t(iy * nl + ix)];
                T s = 0;
                s += at(y - l, x) + at(y + l, x);
                s += at(y, x - l) + at(y, x + l);
                T t = std::fma(-T(4), cur[c], s);
                t = std::fma(h2, g, t);
                nxt[c] = std::fma(wp, t, cur[c]);
                ++g_relax_updates;
            } else {
                // interpolation of the previous variations on the lattice of the node's own subdomain
                int64_t c0[2], c1[2];
                T wl[2], wh[2];
                const int64_t pp[2] = {y, x};
                for (int a = 0; a < 2; ++a) {
                    const bool high = pp[a] >= N / 2;
                    const int64_t t = high ? N - 1 - pp[a] : pp[a];
                    const int64_t i0 = t / l;
                    wh[a] = T(double(t - i0 * l) / double(l));
                    wl[a] = T(1) - wh[a];
                    c0[a] = high ? N - 1 - i0 * l : i0 * l;
                    c1[a] = high ? N - 1 - (i0 + 1) * l : (i0 + 1) * l;
                }
                T acc = 0;
                for (int cy = 0; cy < 2; ++cy)
                    for (int cx = 0; cx < 2; ++cx) {
                        const T wy = cy ? wh[0] : wl[0], wx = cx ? wh[1] : wl[1];
                        if (wy == T(0) || wx == T(0)) continue;
                        const int64_t qy = cy ? c1[0] : c0[0], qx = cx ? c1[1] : c0[1];
                        acc += (wy * wx) * var[size_t(qy * N + qx)];
                    }
                nxt[c] = cur[c] + acc;
                ++g_move_updates;
            }
        }
    prev.swap(cur);
    cur.swap(nxt);
}

template <class T>
double cycle_P(int64_t N, int levels, double h, double omega, bool central, const int* slv, const int* sit, int slen,
               const T* f, T* u, long max_iters, T* cur_out) {
    int64_t d[2] = {N, N};
    Grid F = make_grid(2, d);
    std::vector<T> r(size_t(N * N), T(0));
    double n2 = residual(F, h, (const T*)nullptr, u, f, r.data());
    std::vector<std::vector<T>> E[2][2];
    p2_restrict_all(N, levels, r.data(), E);
    std::vector<T> cur(size_t(N * N), T(0)), prev(size_t(N * N), T(0)), nxt(size_t(N * N), T(0)), var(size_t(N * N), T(0));
    long done = 0;
    for (int s = 0; s < slen && (max_iters < 0 || done < max_iters); ++s)
        for (int it = 0; it < sit[s] && (max_iters < 0 || done < max_iters); ++it, ++done)
            iteration_P(N, slv[s], h, omega, central, E, cur, prev, nxt, var);
    if (cur_out) std::memcpy(cur_out, cur.data(), sizeof(T) * size_t(N * N));
    for (int64_t i = 0; i < N * N; ++i) u[i] += cur[size_t(i)];
    return std::sqrt(n2);
}

inline bool p2_valid(int64_t N, int levels) {
    if (N < 8 || (N & (N - 1)) != 0 || levels < 1) return false;
    return (int64_t(1) << (levels - 1)) <= N / 2;           // coarsest lattice: {anchor, central point} per half
}

template <class T>
int run_homg_p2(int64_t N, int levels, double h, double omega, int central, const int* slv, const int* sit, int slen,
                const void* f_, void* u_, int ncycles, void* hist_, double* norms) {
    if (!p2_valid(N, levels)) return 1;
    for (int s = 0; s < slen; ++s) if (slv[s] < 0 || slv[s] >= levels || sit[s] < 1) return 2;
    const T* f = (const T*)f_;
    T* u = (T*)u_;
    T* hist = (T*)hist_;
    for (int c = 0; c < ncycles; ++c) {
        double n = cycle_P<T>(N, levels, h, omega, central != 0, slv, sit, slen, f, u, -1, nullptr);
        if (norms) norms[c] = n;
        if (hist) std::memcpy(hist + size_t(c) * size_t(N * N), u, sizeof(T) * size_t(N * N));
    }
    int64_t d[2] = {N, N};
    Grid F = make_grid(2, d);
    if (norms) norms[ncycles] = std::sqrt(residual(F, h, (const T*)nullptr, u, f, (T*)nullptr));
    return 0;
}

}  // namespace

#define DISPATCH(dtype, CALL32, CALL64) ((dtype) == 4 ? (CALL32) : (dtype) == 8 ? (CALL64) : -1)

extern "C" {

// out = A v on interior nodes (0 on the boundary) of a per-level array with mesh width h
int orc_apply_A(int dtype, int nd, const int64_t* dims, double h, const void* k, const void* v, void* out) {
    Grid G = make_grid(nd, dims);
    if (dtype == 4) apply_A<float>(G, h, (const float*)k, (const float*)v, (float*)out);
    else if (dtype == 8) apply_A<double>(G, h, (const double*)k, (const double*)v, (double*)out);
    else return -1;
    return 0;
}

// r = f - A u (nullable r); *norm2 = sum over interior of r^2 accumulated in double
int orc_residual(int dtype, int nd, const int64_t* dims, double h, const void* k, const void* u,
                 const void* f, void* r, double* norm2) {
    Grid G = make_grid(nd, dims);
    double s;
    if (dtype == 4) s = residual<float>(G, h, (const float*)k, (const float*)u, (const float*)f, (float*)r);
    else if (dtype == 8) s = residual<double>(G, h, (const double*)k, (const double*)u, (const double*)f, (double*)r);
    else return -1;
    if (norm2) *norm2 = s;
    return 0;
}

// one damped-Jacobi sweep on a per-level array
int orc_jacobi(int dtype, int nd, const int64_t* dims, double h, const void* k, double omega,
               const void* v, const void* g, void* out) {
    Grid G = make_grid(nd, dims);
    if (dtype == 4) jacobi<float>(G, h, (const float*)k, omega, (const float*)v, (const float*)g, (float*)out);
    else if (dtype == 8) jacobi<double>(G, h, (const double*)k, omega, (const double*)v, (const double*)g, (double*)out);
    else return -1;
    return 0;
}

// full weighting, fine dims -> ((n-1)/2+1) dims
int orc_restrict(int dtype, int nd, const int64_t* dims_fine, const void* in, void* out) {
    Grid F = make_grid(nd, dims_fine);
    for (int a = 0; a < nd; ++a) if ((dims_fine[a] - 1) % 2 != 0 || dims_fine[a] < 3) return 1;
    if (dtype == 4) restrict_fw<float>(F, (const float*)in, (float*)out);
    else if (dtype == 8) restrict_fw<double>(F, (const double*)in, (double*)out);
    else return -1;
    return 0;
}

// multilinear prolongation, coarse dims -> (2(n-1)+1) dims
int orc_prolong(int dtype, int nd, const int64_t* dims_coarse, const void* in, void* out) {
    Grid C = make_grid(nd, dims_coarse);
    if (dtype == 4) prolong<float>(C, (const float*)in, (float*)out);
    else if (dtype == 8) prolong<double>(C, (const double*)in, (double*)out);
    else return -1;
    return 0;
}

int orc_schedule(int kind, int levels, int maxI, int* lv, int* it, int cap) {
    return make_schedule(kind, levels, maxI, lv, it, cap);
}

// ncycles outer HOMG cycles.  alg 0 = literal single-array (L), 1 = per-level (H).
// u is in/out; u_hist (nullable) receives u after every cycle (ncycles x N);
// norms (nullable, ncycles+1) receives ||f - A u||_2 before each cycle and after the last.
int orc_homg(int alg, int dtype, int nd, const int64_t* dims, int levels, double h, const void* k,
             double omega, const int* slv, const int* sit, int slen, const void* f, void* u, int ncycles,
             void* u_hist, double* norms) {
    if (dtype == 4) return run_homg<float>(alg, nd, dims, levels, h, k, omega, slv, sit, slen, f, u, ncycles, u_hist, norms);
    if (dtype == 8) return run_homg<double>(alg, nd, dims, levels, h, k, omega, slv, sit, slen, f, u, ncycles, u_hist, norms);
    return -1;
}

// mixed-precision outer loop: fp64 u, f, k; the correction cycle in fp32 (Algorithm H)
int orc_homg_mixed(int nd, const int64_t* dims, int levels, double h, const double* k, double omega, const int* slv,
                   const int* sit, int slen, const double* f, double* u, int ncycles, double* u_hist, double* norms) {
    return run_homg_mixed(nd, dims, levels, h, k, omega, slv, sit, slen, f, u, ncycles, u_hist, norms);
}

// the first `niters` whole-grid iterations of ONE literal cycle started from u;
// cur_out receives the correction array after those iterations (u is not modified).
int orc_homg_L_partial(int nd, const int64_t* dims, int levels, double h, const double* k, double omega,
                       const int* slv, const int* sit, int slen, const double* f, const double* u,
                       long niters, double* cur_out) {
    Hier<double> H;
    if (!build_hier<double>(H, nd, dims, levels, h, k)) return 1;
    std::vector<double> uu(u, u + H.G[0].size());
    cycle_L<double>(H, omega, slv, sit, slen, f, uu.data(), niters, cur_out);
    return 0;
}

int orc_vcycle(int dtype, int nd, const int64_t* dims, int levels, double h, const void* k, double omega,
               int eta1, int eta2, const void* f, void* u, int ncycles, void* u_hist, double* norms) {
    if (dtype == 4) return run_vcycle<float>(nd, dims, levels, h, k, omega, eta1, eta2, f, u, ncycles, u_hist, norms);
    if (dtype == 8) return run_vcycle<double>(nd, dims, levels, h, k, omega, eta1, eta2, f, u, ncycles, u_hist, norms);
    return -1;
}

// dense LU solve of A u = f (double), u = 0 on the boundary
int orc_dense_solve(int nd, const int64_t* dims, double h, const double* k, const double* f, double* u) {
    Grid G = make_grid(nd, dims);
    return dense_solve<double>(G, h, k, f, u) ? 0 : 1;
}

// dense matrix (row-major N x N over interior nodes in C order); returns N
int64_t orc_assemble(int nd, const int64_t* dims, double h, const double* k, double* A, int64_t cap) {
    Grid G = make_grid(nd, dims);
    int64_t N = interior_count(G);
    if (!A) return N;
    if (cap < N * N) return -N;
    std::vector<double> M;
    assemble<double>(G, h, k, M);
    std::memcpy(A, M.data(), sizeof(double) * N * N);
    return N;
}

// ---- Algorithm P (section 3, power-of-two grids; R19) ----
// ncycles outer cycles on an N x N grid, N = 2^k, levels <= k.  central = 0 leaves out the central points (ablation pin).
int orc_homg_p2(int dtype, int64_t N, int levels, double h, double omega, int central, const int* slv, const int* sit,
                int slen, const void* f, void* u, int ncycles, void* u_hist, double* norms) {
    if (dtype == 4) return run_homg_p2<float>(N, levels, h, omega, central, slv, sit, slen, f, u, ncycles, u_hist, norms);
    if (dtype == 8) return run_homg_p2<double>(N, levels, h, omega, central, slv, sit, slen, f, u, ncycles, u_hist, norms);
    return -1;
}
// the correction array after the first `niters` whole-grid iterations of one cycle (u is not modified)
int orc_homg_p2_partial(int64_t N, int levels, double h, double omega, int central, const int* slv, const int* sit, int slen,
                        const double* f, const double* u, long niters, double* cur_out) {
    if (!p2_valid(N, levels)) return 1;
    std::vector<double> uu(u, u + N * N);
    cycle_P<double>(N, levels, h, omega, central != 0, slv, sit, slen, f, uu.data(), niters, cur_out);
    return 0;
}
// mask[y*N+x] = 1 where node (y, x) is marked at level m (boundary nodes included)
int orc_p2_marked(int64_t N, int m, int central, unsigned char* mask) {
    P2Lattice Lt{N, int64_t(1) << m, central != 0};
    for (int64_t y = 0; y < N; ++y)
        for (int64_t x = 0; x < N; ++x) {
            int a;
            mask[y * N + x] = (Lt.on(y, &a) && Lt.on(x, &a)) ? 1 : 0;
        }
    return 0;
}
// one iteration at level m with source 0 from (cur, prev): out = next iterate.  With cur = d, prev = 0 the non-marked
// nodes of `out` hold d + (interpolant of d on their subdomain's lattice): the interpolation operator alone.
int orc_p2_iteration(int64_t N, int levels, int m, double h, double omega, int central, const double* r, const double* cur,
                     const double* prev, double* out) {
    if (!p2_valid(N, levels) || m < 0 || m >= levels) return 1;
    std::vector<std::vector<double>> E[2][2];
    p2_restrict_all<double>(N, levels, r, E);
    std::vector<double> c(cur, cur + N * N), p(prev, prev + N * N), n(size_t(N * N), 0.0), v(size_t(N * N), 0.0);
    iteration_P<double>(N, m, h, omega, central != 0, E, c, p, n, v);
    std::memcpy(out, c.data(), sizeof(double) * size_t(N * N));
    return 0;
}
// the restricted source of level m on the lattice anchored at (ay, ax): (N/2^m + 1)^2 entries indexed from the anchor
int orc_p2_restrict(int64_t N, int levels, int m, int ay, int ax, const double* r, double* out) {
    if (!p2_valid(N, levels) || m < 0 || m >= levels) return 1;
    std::vector<std::vector<double>> E[2][2];
    p2_restrict_all<double>(N, levels, r, E);
    std::memcpy(out, E[ay][ax][m].data(), sizeof(double) * E[ay][ax][m].size());
    return 0;
}

void orc_counters(unsigned long long* relax, unsigned long long* moves, int reset) {
    if (relax) *relax = g_relax_updates;
    if (moves) *moves = g_move_updates;
    if (reset) { g_relax_updates = 0; g_move_updates = 0; }
}

}  // extern "C"
