// Host set-up for the Landau Jacobian path: quadtree leaves -> node lattice,
// hanging-node constraints and their closure, DOF numbering, CSR pattern of A1, deterministic
// gather lists, integration points and basis tabulations.  PAPER.md L101 (inputs of Alg. 1),
// L165 (metadata built once on the CPU), L297 (constrained DOFs interpolate to 4 DOFs for Q3).
// Conventions: include/landau.h.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <map>
#include <unordered_map>

#include "landau_internal.h"

namespace landau {
namespace {

using Key = uint64_t;
inline Key leaf_key(int l, int64_t i, int64_t j) { return (Key(l) << 56) | (Key(i) << 28) | Key(j); }
inline Key node_key(int64_t R, int64_t Z) { return (Key(Z) << 32) | Key(R); }  // sorts by (Z, R)
inline int64_t node_R(Key k) { return int64_t(k & 0xffffffffu); }
inline int64_t node_Z(Key k) { return int64_t(k >> 32); }

// 1-D Lagrange basis on the p+1 equispaced nodes t = 0..p, value at t.
void lagrange_nodes(int p, double t, double *w) {
    for (int a = 0; a <= p; ++a) {
        double v = 1.0;
        for (int b = 0; b <= p; ++b)
            if (b != a) v *= (t - b) / double(a - b);
        w[a] = v;
    }
}

// Values and derivatives on [-1,1] (nodes -1 + 2a/p) at x.
void lagrange_ref(int p, double x, double *val, double *der) {
    double nd[4];
    for (int a = 0; a <= p; ++a) nd[a] = -1.0 + 2.0 * a / p;
    for (int a = 0; a <= p; ++a) {
        double v = 1.0, d = 0.0;
        for (int b = 0; b <= p; ++b)
            if (b != a) v *= (x - nd[b]) / (nd[a] - nd[b]);
        for (int c = 0; c <= p; ++c) {
            if (c == a) continue;
            double t = 1.0 / (nd[a] - nd[c]);
            for (int b = 0; b <= p; ++b)
                if (b != a && b != c) t *= (x - nd[b]) / (nd[a] - nd[b]);
            d += t;
        }
        val[a] = v;
        der[a] = d;
    }
}

// Gauss-Legendre rule with n = 3 or 4 points, closed forms, abscissae ascending.
void gauss_legendre(int n, double *x, double *w) {
    if (n == 3) {
        double a = std::sqrt(3.0 / 5.0);
        x[0] = -a; x[1] = 0.0; x[2] = a;
        w[0] = 5.0 / 9.0; w[1] = 8.0 / 9.0; w[2] = 5.0 / 9.0;
    } else {
        double t = (2.0 / 7.0) * std::sqrt(6.0 / 5.0);
        double a = std::sqrt(3.0 / 7.0 - t), b = std::sqrt(3.0 / 7.0 + t);
        double wa = (18.0 + std::sqrt(30.0)) / 36.0, wb = (18.0 - std::sqrt(30.0)) / 36.0;
        x[0] = -b; x[1] = -a; x[2] = a; x[3] = b;
        w[0] = wb; w[1] = wa; w[2] = wa; w[3] = wb;
    }
}

struct Term { Key node; double w; };
using Row = std::vector<Term>;

}  // namespace

int build_host_space(const landau_mesh &mesh, int order, HostSpace &hs, std::string &err) {
    const int p = order;
    if (p != 2 && p != 3) { err = "order must be 2 or 3"; return LANDAU_EINVAL; }
    if (mesh.ncells < 1 || mesh.nbr < 1 || mesh.nbz < 1 || !mesh.level || !mesh.ir || !mesh.iz) {
        err = "empty mesh"; return LANDAU_EINVAL;
    }
    if (!(mesh.rmax > mesh.rmin) || !(mesh.zmax > mesh.zmin) || mesh.rmin < 0.0) {
        err = "domain must have rmin >= 0 and positive extent"; return LANDAU_EINVAL;
    }
    const int64_t Ne = mesh.ncells;
    const int np1 = p + 1, Nb = np1 * np1, Nq = Nb;
    int Lmax = 0;
    for (int64_t e = 0; e < Ne; ++e) {
        if (mesh.level[e] < 0 || mesh.level[e] > 20) { err = "leaf level out of range"; return LANDAU_EINVAL; }
        Lmax = std::max(Lmax, int(mesh.level[e]));
    }

    // ---- leaves: uniqueness, bounds, coverage --------------------------------------------------
    std::unordered_map<Key, int32_t> leaves;
    leaves.reserve(size_t(Ne) * 2);
    long double area = 0;  // in units of level-Lmax cells
    for (int64_t e = 0; e < Ne; ++e) {
        int l = mesh.level[e];
        int64_t i = mesh.ir[e], j = mesh.iz[e];
        if (i < 0 || j < 0 || i >= (int64_t(mesh.nbr) << l) || j >= (int64_t(mesh.nbz) << l)) {
            err = "leaf outside the domain"; return LANDAU_EINVAL;
        }
        if (!leaves.emplace(leaf_key(l, i, j), int32_t(e)).second) { err = "duplicate leaf"; return LANDAU_EINVAL; }
        area += (long double)(int64_t(1) << (2 * (Lmax - l)));
    }
    if (area != (long double)mesh.nbr * mesh.nbz * (long double)(int64_t(1) << (2 * Lmax))) {
        err = "leaves do not tile the domain"; return LANDAU_EINVAL;
    }
    for (int64_t e = 0; e < Ne; ++e) {  // no leaf may be an ancestor of another (with equal area => exact tiling)
        int l = mesh.level[e];
        int64_t i = mesh.ir[e], j = mesh.iz[e];
        for (int a = l - 1; a >= 0; --a) {
            i >>= 1; j >>= 1;
            if (leaves.count(leaf_key(a, i, j))) { err = "overlapping leaves"; return LANDAU_EINVAL; }
        }
    }

    // ---- hanging nodes ----------------------------------------------------------------------
    // Lattice unit = node spacing of a level-Lmax cell; a level-l cell has node spacing H = 2^(Lmax-l).
    std::map<Key, Row> constraint;
    const int di4[4] = {-1, 1, 0, 0}, dj4[4] = {0, 0, -1, 1};
    for (int64_t e = 0; e < Ne; ++e) {
        const int l = mesh.level[e];
        const int64_t i = mesh.ir[e], j = mesh.iz[e];
        const int64_t H = int64_t(1) << (Lmax - l), Hc = 2 * H;
        for (int f = 0; f < 4; ++f) {
            const int64_t ni = i + di4[f], nj = j + dj4[f];
            if (ni < 0 || nj < 0 || ni >= (int64_t(mesh.nbr) << l) || nj >= (int64_t(mesh.nbz) << l)) continue;
            if (leaves.count(leaf_key(l, ni, nj))) continue;
            if (l > 0 && leaves.count(leaf_key(l - 1, ni >> 1, nj >> 1))) {
                const int64_t I = ni >> 1, J = nj >> 1;
                for (int a = 0; a <= p; ++a) {
                    int64_t R, Z, num;  // num/Hc = position on the coarse edge in coarse node units
                    Key par[4];
                    if (di4[f] != 0) {
                        R = (i + (di4[f] > 0 ? 1 : 0)) * p * H; Z = j * p * H + a * H; num = Z - J * p * Hc;
                        for (int b = 0; b <= p; ++b) par[b] = node_key(R, J * p * Hc + b * Hc);
                    } else {
                        Z = (j + (dj4[f] > 0 ? 1 : 0)) * p * H; R = i * p * H + a * H; num = R - I * p * Hc;
                        for (int b = 0; b <= p; ++b) par[b] = node_key(I * p * Hc + b * Hc, Z);
                    }
                    if (num % Hc == 0) continue;  // coincides with a coarse node: shared, not hanging
                    double w[4];
                    lagrange_nodes(p, double(num) / double(Hc), w);
                    Row row;
                    for (int b = 0; b <= p; ++b) row.push_back({par[b], w[b]});
                    constraint[node_key(R, Z)] = row;
                }
                continue;
            }
            // otherwise the neighbour must be exactly one level finer (2:1 face balance)
            const int64_t ci = 2 * ni + (di4[f] < 0 ? 1 : 0), cj = 2 * nj + (dj4[f] < 0 ? 1 : 0);
            const int64_t ci2 = ci + (di4[f] == 0 ? 1 : 0), cj2 = cj + (dj4[f] == 0 ? 1 : 0);
            if (!leaves.count(leaf_key(l + 1, ci, cj)) || !leaves.count(leaf_key(l + 1, ci2, cj2))) {
                err = "mesh is not 2:1 face balanced"; return LANDAU_EINVAL;
            }
        }
    }

    // ---- closure: expand parents that are themselves hanging (coarser constraints first) -----
    std::map<Key, Row> closed;
    std::vector<Key> order_keys;
    for (auto &kv : constraint) order_keys.push_back(kv.first);
    for (int pass = 0; pass < 64 && !order_keys.empty(); ++pass) {
        std::vector<Key> pending;
        for (Key k : order_keys) {
            const Row &row = constraint[k];
            bool ready = true;
            for (const Term &t : row)
                if (constraint.count(t.node) && !closed.count(t.node)) ready = false;
            if (!ready) { pending.push_back(k); continue; }
            std::map<Key, double> acc;
            for (const Term &t : row) {
                auto it = closed.find(t.node);
                if (it == closed.end()) acc[t.node] += t.w;
                else for (const Term &u : it->second) acc[u.node] += t.w * u.w;
            }
            Row out;
            for (auto &kv : acc) out.push_back({kv.first, kv.second});
            closed[k] = out;
        }
        if (pending.size() == order_keys.size()) { err = "cyclic hanging-node constraints"; return LANDAU_EINVAL; }
        order_keys.swap(pending);
    }

    // ---- DOF numbering: free nodes by ascending (Z, R) ------------------------------------------
    std::vector<Key> nodes;
    nodes.reserve(size_t(Ne) * Nb);
    for (int64_t e = 0; e < Ne; ++e) {
        const int64_t H = int64_t(1) << (Lmax - mesh.level[e]);
        for (int az = 0; az <= p; ++az)
            for (int ar = 0; ar <= p; ++ar)
                nodes.push_back(node_key(int64_t(mesh.ir[e]) * p * H + ar * H, int64_t(mesh.iz[e]) * p * H + az * H));
    }
    std::vector<Key> cell_nodes = nodes;  // [Ne*Nb], local order
    std::sort(nodes.begin(), nodes.end());
    nodes.erase(std::unique(nodes.begin(), nodes.end()), nodes.end());
    std::vector<Key> free_nodes;
    for (Key k : nodes)
        if (!closed.count(k)) free_nodes.push_back(k);
    const int64_t n = int64_t(free_nodes.size());
    auto dof_of = [&](Key k) { return int32_t(std::lower_bound(free_nodes.begin(), free_nodes.end(), k) - free_nodes.begin()); };

    hs.p = p; hs.Nq = Nq; hs.Nb = Nb; hs.Ne = Ne; hs.N = Ne * Nq; hs.n = n;
    const double hr0 = (mesh.rmax - mesh.rmin) / mesh.nbr, hz0 = (mesh.zmax - mesh.zmin) / mesh.nbz;
    const double ur = hr0 / (double(p) * double(int64_t(1) << Lmax)), uz = hz0 / (double(p) * double(int64_t(1) << Lmax));
    hs.dof_r.resize(n); hs.dof_z.resize(n);
    for (int64_t d = 0; d < n; ++d) {
        hs.dof_r[d] = mesh.rmin + double(node_R(free_nodes[d])) * ur;
        hs.dof_z[d] = mesh.zmin + double(node_Z(free_nodes[d])) * uz;
    }

    // ---- local node -> free DOFs ----------------------------------------------------------------
    hs.lptr.assign(size_t(Ne) * Nb + 1, 0);
    hs.ldof.clear(); hs.lw.clear();
    for (size_t t = 0; t < cell_nodes.size(); ++t) {
        auto it = closed.find(cell_nodes[t]);
        if (it == closed.end()) {
            hs.ldof.push_back(dof_of(cell_nodes[t])); hs.lw.push_back(1.0);
        } else {
            for (const Term &u : it->second) { hs.ldof.push_back(dof_of(u.node)); hs.lw.push_back(u.w); }
        }
        hs.lptr[t + 1] = int32_t(hs.ldof.size());
    }

    // ---- integration points and weights (reading Q2) -----------------------------------------
    double xg[4], wg[4];
    gauss_legendre(np1, xg, wg);
    hs.r.resize(hs.N); hs.z.resize(hs.N); hs.w_in.resize(hs.N); hs.w_out.resize(hs.N);
    hs.invJ.resize(size_t(Ne) * 2);
    const double two_pi = 6.283185307179586476925286766559;
    for (int64_t e = 0; e < Ne; ++e) {
        const double sc = 1.0 / double(int64_t(1) << mesh.level[e]);
        const double hr = hr0 * sc, hz = hz0 * sc;
        const double r0 = mesh.rmin + mesh.ir[e] * hr, z0 = mesh.zmin + mesh.iz[e] * hz;
        hs.invJ[2 * e] = 2.0 / hr; hs.invJ[2 * e + 1] = 2.0 / hz;
        const double detJ = 0.25 * hr * hz;
        for (int qz = 0; qz <= p; ++qz)
            for (int qr = 0; qr <= p; ++qr) {
                const int64_t gi = e * Nq + qz * np1 + qr;
                hs.r[gi] = r0 + 0.5 * (xg[qr] + 1.0) * hr;
                hs.z[gi] = z0 + 0.5 * (xg[qz] + 1.0) * hz;
                hs.w_in[gi] = wg[qr] * wg[qz] * detJ * hs.r[gi];
                hs.w_out[gi] = two_pi * hs.w_in[gi];
            }
    }

    // ---- tabulations B, E (L101) --------------------------------------------------------------
    double val[4][4], der[4][4];
    for (int q = 0; q <= p; ++q) lagrange_ref(p, xg[q], val[q], der[q]);
    hs.B.assign(size_t(Nq) * Nb, 0.0); hs.E0 = hs.B; hs.E1 = hs.B;
    for (int qz = 0; qz <= p; ++qz)
        for (int qr = 0; qr <= p; ++qr)
            for (int az = 0; az <= p; ++az)
                for (int ar = 0; ar <= p; ++ar) {
                    const size_t t = size_t(qz * np1 + qr) * Nb + (az * np1 + ar);
                    hs.B[t] = val[qr][ar] * val[qz][az];
                    hs.E0[t] = der[qr][ar] * val[qz][az];
                    hs.E1[t] = val[qr][ar] * der[qz][az];
                }

    // ---- CSR pattern of A1 and the gather lists (deterministic assembly, north_star (3)) -------
    // Every (e,a,b) with expansions (row dof, wa) x (col dof, wb) contributes wa*wb*C_e[a][b] to
    // entry (row, col).  Sort by (row, col, source index): the summation order is fixed.
    struct Coo { int32_t row, col, src; double w; };
    std::vector<Coo> coo;
    coo.reserve(size_t(Ne) * Nb * Nb * 2);
    for (int64_t e = 0; e < Ne; ++e)
        for (int a = 0; a < Nb; ++a)
            for (int b = 0; b < Nb; ++b) {
                const int32_t src = int32_t((e * Nb + a) * Nb + b);
                for (int32_t ta = hs.lptr[e * Nb + a]; ta < hs.lptr[e * Nb + a + 1]; ++ta)
                    for (int32_t tb = hs.lptr[e * Nb + b]; tb < hs.lptr[e * Nb + b + 1]; ++tb)
                        coo.push_back({hs.ldof[ta], hs.ldof[tb], src, hs.lw[ta] * hs.lw[tb]});
            }
    std::sort(coo.begin(), coo.end(), [](const Coo &x, const Coo &y) {
        if (x.row != y.row) return x.row < y.row;
        if (x.col != y.col) return x.col < y.col;
        return x.src < y.src;
    });
    hs.rowptr.assign(n + 1, 0);
    hs.colidx.clear(); hs.gptr.clear(); hs.gidx.clear(); hs.gw.clear();
    for (size_t t = 0; t < coo.size(); ++t) {
        if (t == 0 || coo[t].row != coo[t - 1].row || coo[t].col != coo[t - 1].col) {
            hs.colidx.push_back(coo[t].col);
            hs.gptr.push_back(int32_t(hs.gidx.size()));
            hs.rowptr[coo[t].row + 1]++;
        }
        hs.gidx.push_back(coo[t].src);
        hs.gw.push_back(coo[t].w);
    }
    hs.gptr.push_back(int32_t(hs.gidx.size()));
    for (int64_t d = 0; d < n; ++d) hs.rowptr[d + 1] += hs.rowptr[d];
    hs.nnz = int64_t(hs.colidx.size());

    // element-vector gather (C(f)): dof d <- (e*Nb + a, weight)
    struct Cv { int32_t dof, src; double w; };
    std::vector<Cv> cv;
    for (int64_t t = 0; t < Ne * Nb; ++t)
        for (int32_t u = hs.lptr[t]; u < hs.lptr[t + 1]; ++u) cv.push_back({hs.ldof[u], int32_t(t), hs.lw[u]});
    std::sort(cv.begin(), cv.end(), [](const Cv &x, const Cv &y) { return x.dof != y.dof ? x.dof < y.dof : x.src < y.src; });
    hs.cptr.assign(n + 1, 0); hs.cidx.clear(); hs.cw.clear();
    for (const Cv &c : cv) { hs.cptr[c.dof + 1]++; hs.cidx.push_back(c.src); hs.cw.push_back(c.w); }
    for (int64_t d = 0; d < n; ++d) hs.cptr[d + 1] += hs.cptr[d];
    return LANDAU_OK;
}

}  // namespace landau
