// Symbolic layer of the complementary-operator two-site DMRG (host, integers and 16x16 matrices only).
//
// The paper fixes WHAT is computed (H of PAPER.md:52-68 Eq. 1-5, MPS of Eq. 14) and defers HOW to its refs
// [44,50,60]; the algorithm restated here is DESIGN.md "Algorithm":
//   H = H_A + H_B + sum_{P in A}(a+_P S_P^B + h.c.) + sum_{P in B}(a+_P S_P^A + h.c.)
//       + sum_{P<Q in A}(A_PQ P_PQ^B + h.c.) + sum_{P,S in A} B_PS Q_PS^B                       (bipartition identity)
//   S_P^X = sum_Q 1/2 t_PQ a_Q + sum_QRS v_PQRS a+_Q a_R a_S,  P_PQ^X = sum_RS v_PQRS a_R a_S,
//   Q_PS^X = sum_QR (v_PQRS - v_PQSR) a+_Q a_R.
// Every enlarged-block operator and every H_eff term is generated mechanically from these identities as a list of
// (coefficient, ordered factors) and brought into chain order with the Jordan-Wigner sign rule; nothing is
// hand-enumerated.  Stored operator kinds: H, C = a+_P, St = (S_P)^T, A = a+_P a+_Q (P<Q), B = a+_P a_S,
// Pt = (P_PQ)^T (P<Q), Q = Q_PS, and the one-index linear combinations U_{P;RS} = sum_Q w_PQRS a+_Q,
// V_{P;QR} = sum_S w_PQRS a+_S (w = v_PQRS - v_PQSR) that keep the growth of S_P at O(1) pieces per operator.
#pragma once
#include <array>
#include <cstdint>
#include <cstring>
#include <vector>

namespace dmrg {

static const int SITE_QN[4] = {0, 1, 1, 2};    // particle number of |0>, |dn>, |up>, |up dn>
static const int SITE_QS[4] = {0, -1, 1, 0};   // 2Sz

inline int spin_of(int P) { return (P & 1) == 0 ? 1 : -1; }   // spin orbital P = 2p + [down]

struct Ham {
    int k = 0;
    std::vector<double> h, eri;
    double t(int P, int Q) const { return ((P & 1) == (Q & 1)) ? h[(size_t)(P >> 1) * k + (Q >> 1)] : 0.0; }
    // v_PQRS = (ps|qr) d(sP,sS) d(sQ,sR):  H = sum t a+a + 1/2 sum v a+_P a+_Q a_R a_S
    double v(int P, int Q, int R, int S) const {
        if ((P & 1) != (S & 1) || (Q & 1) != (R & 1)) return 0.0;
        return eri[(((size_t)(P >> 1) * k + (S >> 1)) * k + (Q >> 1)) * k + (R >> 1)];
    }
    double w(int P, int Q, int R, int S) const { return v(P, Q, R, S) - v(P, Q, S, R); }
};

// small dense square matrix (n = 4 for one site, 16 for the two-site dot, state index 4*s_i + s_j)
struct Mat {
    int n = 0;
    std::vector<double> a;
    Mat() {}
    explicit Mat(int n_) : n(n_), a((size_t)n_ * n_, 0.0) {}
    double& operator()(int i, int j) { return a[(size_t)i * n + j]; }
    double operator()(int i, int j) const { return a[(size_t)i * n + j]; }
    static Mat eye(int n);
    Mat T() const;
    Mat operator*(const Mat& o) const;
    void axpy(double c, const Mat& o);
    bool any() const;
};

enum Kind : int { K_I = 0, K_H, K_C, K_St, K_A, K_B, K_Pt, K_Q, K_U, K_V, K_NKINDS };
extern const int KIND_PAR[K_NKINDS];

struct Label {
    int kind = K_I, a = 0, b = 0, c = 0;
    uint32_t key() const { return ((uint32_t)kind << 24) | ((uint32_t)a << 16) | ((uint32_t)b << 8) | (uint32_t)c; }
    bool operator==(const Label& o) const { return key() == o.key(); }
};
inline Label L0(int kind) { Label l; l.kind = kind; return l; }
inline Label L1(int kind, int a) { Label l; l.kind = kind; l.a = a; return l; }
inline Label L2(int kind, int a, int b) { Label l; l.kind = kind; l.a = a; l.b = b; return l; }
inline Label L3(int kind, int a, int b, int c) { Label l; l.kind = kind; l.a = a; l.b = b; l.c = c; return l; }

// quantum-number shift (dN, d2Sz) of the operator a label names (untransposed)
void op_shift(const Label& l, int& dn, int& ds);

// the "dot": one or two explicit sites with their 4^n-dimensional local space
struct Dot {
    const Ham* ham = nullptr;
    std::vector<int> sites;       // spatial orbitals
    std::vector<int> so;          // their spin orbitals, ascending
    int n = 0;                    // 4 or 16
    std::vector<int> qn, qs;      // quantum numbers of the local states
    std::vector<Mat> c_;          // annihilators, indexed like `so`
    Dot(const Ham* ham, const std::vector<int>& sites);
    bool has(int P) const;
    const Mat& c(int P) const;    // a_P
    Mat cd(int P) const { return c(P).T(); }
    Mat H() const;                // all terms of H with every index on the dot
    Mat S(int P) const;           // S_P^dot
    int parity(const Mat& m) const;   // fermion parity (0/1) from the non-zero pattern
};

// one factor of a symbolic product: a stored operator of the left or right block, or an explicit dot matrix
struct Factor {
    int type = 0;        // 0 = block operator, 1 = dot matrix
    char side = 'L';     // 'L' / 'R' for block operators
    Label label;
    bool trans = false;
    Mat m;
};
struct Term {
    double coef = 1.0;
    std::vector<Factor> f;
};
typedef std::vector<Term> Expr;

// a term in chain order  L . dot . R  (absent block factors are the identity)
struct NTerm {
    double coef = 0.0;
    bool hasL = false, hasR = false;
    Label L, R;
    bool transL = false, transR = false;
    Mat dm;              // dot matrix (identity if no dot factor)
};

Term adjoint(const Term& t);
// chain: order of the parts, e.g. "Ld", "dR", "LdR"; returns the term in that order with the reordering sign
NTerm normalise(const Term& t, const char* chain, const Dot& dot);

struct BlockInfo {          // what the generator needs to know about the block X it enlarges
    char side;
    std::vector<int> inside;     // spin orbitals inside X, ascending
    bool (*has_op)(const void* blk, const Label& l);
    const void* blk;
};

// expressions of operators on X u dot in terms of (operators of X) x (dot matrices)
struct Gen {
    const Ham& ham;
    const Dot& dot;
    BlockInfo X;
    std::vector<char> in_x;      // indexed by spin orbital
    Gen(const Ham& ham, const BlockInfo& X, const Dot& dot);
    Factor bf(const Label& l, bool trans = false) const;
    Factor df(const Mat& m) const;
    bool inX(int P) const { return in_x[P] != 0; }
    void Pc(int P, int Q, double& coef, Factor& f) const;   // P_PQ^X as coef * factor
    void Qc(int P, int S, double& coef, Factor& f) const;
    Expr cre(int P) const;
    Expr ann(int P) const;
    static Expr mul(const Expr& a, const Expr& b);
    Expr A(int P, int Q) const;
    Expr B(int P, int S) const;
    Expr H() const;
    Expr S(int P) const;         // S_P^{X u dot}, P outside
};

}  // namespace dmrg
