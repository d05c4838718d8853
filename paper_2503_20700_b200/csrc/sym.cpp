// Symbolic layer: see sym.hpp.
#include "sym.hpp"

#include <algorithm>
#include <cassert>
#include <stdexcept>

namespace dmrg {

const int KIND_PAR[K_NKINDS] = {0, 0, 1, 1, 0, 0, 0, 0, 1, 1};

Mat Mat::eye(int n) {
    Mat m(n);
    for (int i = 0; i < n; ++i) m(i, i) = 1.0;
    return m;
}
Mat Mat::T() const {
    Mat m(n);
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) m(j, i) = (*this)(i, j);
    return m;
}
Mat Mat::operator*(const Mat& o) const {
    assert(n == o.n);
    Mat m(n);
    for (int i = 0; i < n; ++i)
        for (int l = 0; l < n; ++l) {
            const double x = (*this)(i, l);
            if (x == 0.0) continue;
            for (int j = 0; j < n; ++j) m(i, j) += x * o(l, j);
        }
    return m;
}
void Mat::axpy(double c, const Mat& o) {
    for (size_t i = 0; i < a.size(); ++i) a[i] += c * o.a[i];
}
bool Mat::any() const {
    for (double x : a)
        if (x != 0.0) return true;
    return false;
}

void op_shift(const Label& l, int& dn, int& ds) {
    switch (l.kind) {
        case K_I: case K_H: dn = 0; ds = 0; return;
        case K_C: case K_St: dn = 1; ds = spin_of(l.a); return;
        case K_A: case K_Pt: dn = 2; ds = spin_of(l.a) + spin_of(l.b); return;
        case K_B: dn = 0; ds = spin_of(l.a) - spin_of(l.b); return;
        case K_Q: dn = 0; ds = spin_of(l.b) - spin_of(l.a); return;
        case K_U: dn = 1; ds = spin_of(l.b) + spin_of(l.c) - spin_of(l.a); return;   // U_{P;RS}: spin of Q
        case K_V: dn = 1; ds = spin_of(l.a) + spin_of(l.b) - spin_of(l.c); return;   // V_{P;QR}: spin of S
    }
    throw std::logic_error("op_shift: bad kind");
}

// ---------------------------------------------------------------------------------------------------------------
// Dot
// ---------------------------------------------------------------------------------------------------------------
static Mat site_ann(int down) {     // basis |0>,|dn>,|up>,|up dn> with |up dn> = a+_up a+_dn |0>  (reading S3)
    Mat m(4);
    if (!down) { m(0, 2) = 1.0; m(1, 3) = 1.0; }      // a_up
    else       { m(0, 1) = 1.0; m(2, 3) = -1.0; }     // a_dn
    return m;
}
static Mat kron(const Mat& x, const Mat& y) {
    Mat m(x.n * y.n);
    for (int i = 0; i < x.n; ++i)
        for (int j = 0; j < x.n; ++j) {
            const double v = x(i, j);
            if (v == 0.0) continue;
            for (int a = 0; a < y.n; ++a)
                for (int b = 0; b < y.n; ++b) m(i * y.n + a, j * y.n + b) = v * y(a, b);
        }
    return m;
}

Dot::Dot(const Ham* ham_, const std::vector<int>& sites_) : ham(ham_), sites(sites_) {
    const int ns = (int)sites.size();
    n = 1;
    for (int i = 0; i < ns; ++i) n *= 4;
    Mat F(4);                                   // site parity operator (Jordan-Wigner string)
    F(0, 0) = 1.0; F(1, 1) = -1.0; F(2, 2) = -1.0; F(3, 3) = 1.0;
    for (int idx = 0; idx < ns; ++idx)
        for (int x = 0; x < 2; ++x) {
            Mat m = Mat::eye(1);
            for (int j = 0; j < ns; ++j) m = kron(m, j == idx ? site_ann(x) : (j < idx ? F : Mat::eye(4)));
            so.push_back(2 * sites[idx] + x);
            c_.push_back(m);
        }
    qn.assign(n, 0);
    qs.assign(n, 0);
    for (int st = 0; st < n; ++st) {
        int x = st;
        for (int j = 0; j < ns; ++j) {
            qn[st] += SITE_QN[x % 4];
            qs[st] += SITE_QS[x % 4];
            x /= 4;
        }
    }
}
bool Dot::has(int P) const { return std::find(so.begin(), so.end(), P) != so.end(); }
const Mat& Dot::c(int P) const {
    for (size_t i = 0; i < so.size(); ++i)
        if (so[i] == P) return c_[i];
    throw std::logic_error("Dot::c: orbital not on the dot");
}
Mat Dot::H() const {
    Mat m(n);
    for (int P : so)
        for (int Q : so) {
            const double t = ham->t(P, Q);
            if (t != 0.0) m.axpy(t, cd(P) * c(Q));
            for (int R : so)
                for (int S : so) {
                    const double v = ham->v(P, Q, R, S);
                    if (v != 0.0) m.axpy(0.5 * v, cd(P) * cd(Q) * c(R) * c(S));
                }
        }
    return m;
}
Mat Dot::S(int P) const {
    Mat m(n);
    for (int Q : so) {
        const double t = ham->t(P, Q);
        if (t != 0.0) m.axpy(0.5 * t, c(Q));
        for (int R : so)
            for (int S : so) {
                const double v = ham->v(P, Q, R, S);
                if (v != 0.0) m.axpy(v, cd(Q) * c(R) * c(S));
            }
    }
    return m;
}
int Dot::parity(const Mat& m) const {
    int par = -1;
    for (int a = 0; a < n; ++a)
        for (int b = 0; b < n; ++b)
            if (m(a, b) != 0.0) {
                const int p = (qn[a] - qn[b]) & 1;
                if (par >= 0 && par != p) throw std::logic_error("dot matrix of mixed fermion parity");
                par = p;
            }
    return par < 0 ? 0 : par;
}

// ---------------------------------------------------------------------------------------------------------------
// terms
// ---------------------------------------------------------------------------------------------------------------
Term adjoint(const Term& t) {
    Term r;
    r.coef = t.coef;
    for (auto it = t.f.rbegin(); it != t.f.rend(); ++it) {
        Factor f = *it;
        if (f.type == 0) f.trans = !f.trans;
        else f.m = f.m.T();
        r.f.push_back(f);
    }
    return r;
}

NTerm normalise(const Term& t, const char* chain, const Dot& dot) {
    const int nf = (int)t.f.size();
    std::vector<int> part(nf), par(nf), order(nf);
    for (int j = 0; j < nf; ++j) {
        const char tag = t.f[j].type == 0 ? t.f[j].side : 'd';
        const char* pos = std::strchr(chain, tag);
        if (!pos) throw std::logic_error("normalise: factor not on the chain");
        part[j] = (int)(pos - chain);
        par[j] = t.f[j].type == 0 ? KIND_PAR[t.f[j].label.kind] : dot.parity(t.f[j].m);
        order[j] = j;
    }
    double sign = 1.0;
    for (int a = 0; a < nf; ++a)                       // stable bubble sort, sign from odd-odd exchanges
        for (int b = 0; b + 1 < nf - a; ++b)
            if (part[order[b]] > part[order[b + 1]]) {
                if (par[order[b]] && par[order[b + 1]]) sign = -sign;
                std::swap(order[b], order[b + 1]);
            }
    NTerm r;
    r.coef = t.coef * sign;
    bool have_dm = false;
    for (int j : order) {
        const Factor& f = t.f[j];
        if (f.type == 1) {
            r.dm = have_dm ? r.dm * f.m : f.m;
            have_dm = true;
        } else if (f.side == 'L') {
            if (r.hasL) throw std::logic_error("normalise: two factors on L");
            r.hasL = true; r.L = f.label; r.transL = f.trans;
        } else {
            if (r.hasR) throw std::logic_error("normalise: two factors on R");
            r.hasR = true; r.R = f.label; r.transR = f.trans;
        }
    }
    if (!have_dm) r.dm = Mat::eye(dot.n);
    return r;
}

// ---------------------------------------------------------------------------------------------------------------
// generator of enlarged-block operators
// ---------------------------------------------------------------------------------------------------------------
Gen::Gen(const Ham& ham_, const BlockInfo& X_, const Dot& dot_) : ham(ham_), dot(dot_), X(X_) {
    in_x.assign(2 * ham.k, 0);
    for (int P : X.inside) in_x[P] = 1;
}
Factor Gen::bf(const Label& l, bool trans) const {
    Factor f; f.type = 0; f.side = X.side; f.label = l; f.trans = trans;
    return f;
}
Factor Gen::df(const Mat& m) const {
    Factor f; f.type = 1; f.m = m;
    return f;
}
void Gen::Pc(int P, int Q, double& coef, Factor& f) const {
    if (P < Q) { coef = 1.0; f = bf(L2(K_Pt, P, Q), true); }
    else       { coef = -1.0; f = bf(L2(K_Pt, Q, P), true); }
}
void Gen::Qc(int P, int S, double& coef, Factor& f) const { coef = 1.0; f = bf(L2(K_Q, P, S), false); }

Expr Gen::cre(int P) const {
    Term t;
    t.f.push_back(dot.has(P) ? df(dot.cd(P)) : bf(L1(K_C, P)));
    return Expr{t};
}
Expr Gen::ann(int P) const {
    Expr e;
    for (const Term& t : cre(P)) e.push_back(adjoint(t));
    return e;
}
Expr Gen::mul(const Expr& a, const Expr& b) {
    Expr e;
    for (const Term& x : a)
        for (const Term& y : b) {
            Term t;
            t.coef = x.coef * y.coef;
            t.f = x.f;
            t.f.insert(t.f.end(), y.f.begin(), y.f.end());
            e.push_back(t);
        }
    return e;
}
Expr Gen::A(int P, int Q) const {
    assert(P < Q);
    if (inX(P) && inX(Q)) { Term t; t.f.push_back(bf(L2(K_A, P, Q))); return Expr{t}; }
    return mul(cre(P), cre(Q));
}
Expr Gen::B(int P, int S) const {
    if (inX(P) && inX(S)) { Term t; t.f.push_back(bf(L2(K_B, P, S))); return Expr{t}; }
    return mul(cre(P), ann(S));
}
Expr Gen::H() const {
    Expr T, G;
    const bool xin = !X.inside.empty();
    if (xin) { Term t; t.f.push_back(bf(L0(K_H))); T.push_back(t); }
    { Term t; t.f.push_back(df(dot.H())); T.push_back(t); }
    for (int P : X.inside) {                               // a+_P^X S_P^dot
        Mat m = dot.S(P);
        if (m.any()) { Term t; t.f.push_back(bf(L1(K_C, P))); t.f.push_back(df(m)); G.push_back(t); }
    }
    if (xin) {
        for (int P : dot.so) {                             // a+_P^dot S_P^X
            Term t; t.f.push_back(df(dot.cd(P))); t.f.push_back(bf(L1(K_St, P), true)); G.push_back(t);
        }
        for (size_t a = 0; a < dot.so.size(); ++a)         // A^dot_PQ P^X_PQ
            for (size_t b = a + 1; b < dot.so.size(); ++b) {
                const int P = dot.so[a], Q = dot.so[b];
                Term t; Factor f; Pc(P, Q, t.coef, f);
                t.f.push_back(df(dot.cd(P) * dot.cd(Q))); t.f.push_back(f); G.push_back(t);
            }
    }
    for (const Term& t : G) T.push_back(t);
    for (const Term& t : G) T.push_back(adjoint(t));
    if (xin)
        for (int P : dot.so)                               // B^dot_PS Q^X_PS
            for (int S : dot.so) {
                Term t; Factor f; Qc(P, S, t.coef, f);
                t.f.push_back(df(dot.cd(P) * dot.c(S))); t.f.push_back(f); T.push_back(t);
            }
    return T;
}
Expr Gen::S(int P) const {
    Expr T;
    const bool xin = !X.inside.empty();
    if (xin) { Term t; t.f.push_back(bf(L1(K_St, P), true)); T.push_back(t); }
    { Mat m = dot.S(P); if (m.any()) { Term t; t.f.push_back(df(m)); T.push_back(t); } }
    if (!xin) return T;
    for (size_t a = 0; a < dot.so.size(); ++a)             // sum_{Q in X} w_PQRS a+_Q  a_R a_S,  R<S on the dot
        for (size_t b = a + 1; b < dot.so.size(); ++b) {
            const int R = dot.so[a], S_ = dot.so[b];
            const Label l = L3(K_U, P, R, S_);
            if (X.has_op(X.blk, l)) {
                Term t; t.f.push_back(bf(l)); t.f.push_back(df(dot.c(R) * dot.c(S_))); T.push_back(t);
            }
        }
    for (int Q : dot.so) {                                 // a+_Q^dot P^X_PQ
        Term t; Factor f; Pc(P, Q, t.coef, f);
        t.f.push_back(df(dot.cd(Q))); t.f.push_back(f); T.push_back(t);
    }
    for (int S_ : dot.so) {                                // Q^X_PS a_S^dot
        Term t; Factor f; Qc(P, S_, t.coef, f);
        t.f.push_back(f); t.f.push_back(df(dot.c(S_))); T.push_back(t);
    }
    for (int Q : dot.so)                                   // a+_Q^dot a_R^dot sum_{S in X} w_PQRS a_S
        for (int R : dot.so) {
            const Label l = L3(K_V, P, Q, R);
            if (X.has_op(X.blk, l)) {
                Term t; t.f.push_back(df(dot.cd(Q) * dot.c(R))); t.f.push_back(bf(l, true)); T.push_back(t);
            }
        }
    return T;
}

}  // namespace dmrg
