// wl_oracle.cpp — CPU ORACLE for the pressure-projection path.  TEST INFRASTRUCTURE ONLY.
//
// A plain, slow, single-threaded C++17 statement of what the hot path computes, written from the
// paper (/root/reference/PAPER.md, cited as PAPER.md:N) and the problem statement in
// BASELINE.json `north_star` (cited as BJ "..."), before any CUDA kernel existed.  It shares no
// code, header, table or helper with the CUDA library under paper_2304_08159_b200/csrc and
// neither includes the other.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load it.  Build: g++ -O2 -ffp-contract=off -shared -fPIC (no FMA
// contraction, IEEE division).
//
// Parity status of each function (what pins it other than itself: tests/test_oracle_*.py):
//   apply_A        pinned: Kronecker-sum Neumann Laplacian (uniform L), -G^T diag(L) G incidence
//                  form (variable L), symmetry, negative semi-definiteness, A·1 = 0, diag = -D,
//                  cosine eigenvectors with the closed-form eigenvalue.
//   coarsen, restrict_sum, prolong_add
//                  pinned: dense R = P^T and A_c = R·A·P on tiny grids, uniform L -> 2^(n-1),
//                  dyadic-rational L exact in any order.
//   jacobi         pinned: dense x + w D^-1 (A x - b) with the pinned dense A.
//   vcycle         pinned as far as anything external can: dense-matrix multigrid recursion built
//                  in NumPy from the pinned A, R, P (tests/test_oracle_cycle.py).  The cycle's
//                  constants (w = 2/3, 2+2 sweeps, 64 coarse sweeps) are fixed by BJ's text only:
//                  no published value exists for them -> "parity unpinned" by any external number.
//   solve          pinned: converges to the dense pseudo-inverse solution (8^2, 8^3, 12x8, 16^2
//                  with a body) and to the cosine closed form; monotone residual history.
//   divergence, gradient_correct, project
//                  pinned: div(u_out) == b - A p to rounding; max|div u_out| <= tol·max|b| when
//                  converged; -G^T / G incidence forms.
//   solve_pcg      ("Conjugate-Gradient ... within the GMG")
//                  pinned: textbook preconditioned CG written with dense NumPy matrices (the
//                  preconditioner = the dense-matrix V-cycle of tests/test_oracle_cycle.py applied
//                  to unit vectors), iterate by iterate; M^-1-orthogonality of the residuals and
//                  A-conjugacy of the directions; termination on the dense pseudo-inverse solution
//                  in <= rank(A) steps on tiny grids (tests/test_oracle_pcg.py).  The reading
//                  (V-cycle as preconditioner, where the mean is removed, fp64 dot products) is
//                  DESIGN.md section 3 reading 13: the paper gives no detail -> "parity unpinned" by any
//                  value of the paper.
//
//   body_coeff     (the BDIM! row of Table 2)
//                  pinned (tests/test_oracle_body.py): mu0(-1) = 0, mu0(0) = 1/2, mu0(1) = 1, the closed forms
//                  mu0(+-1/2) = 1/2 +- (1/4 + 1/(2 pi)), mu0(d) + mu0(-d) = 1, monotone, contact with 0 and 1
//                  at +-1 (1e-11 at 1e-4 inside), never negative just inside d = -1; exact 0 / 1 at faces
//                  farther than one cell inside / outside a body and 0 on the stored wall planes; the
//                  face-centre convention on a radius-1/2 sphere centred ON a face centre (closed-form
//                  distances of the neighbouring face centres); the lattice sum of 1 - L over each face
//                  family against 4/3 pi R^3 + 4 pi R (1/3 - 2/pi^2); several bodies = the minimum distance;
//                  a torus with faces exactly on its surface, centre line and one cell outside.
//
//   convdiff       (`convdiff!`; "third-order finite volume")
//                  pinned: the face value against Leonard's normalised-variable diagram written independently, exact
//                  point value of any quadratic given by its cell averages, boundedness; the diffusive part
//                  (r(nu=1) - r(nu=0)) against a Kronecker-sum Laplacian with free-slip walls; second-order
//                  convergence to -(u.grad)u + nu lap u of the Taylor-Green field (signs, the 1/2 of the advecting
//                  velocity, every index offset); a step profile advected both ways (upwind direction); mirror and
//                  axis-permutation covariance; momentum conservation (tests/test_oracle_convdiff.py).  The scheme's
//                  details are DESIGN.md section 3 reading 15: the paper prints none -> "parity unpinned" by any value
//                  of the paper.
//
// Notation: n = ndim in {2,3}; N = (N_0..N_{n-1}), axis 0 unit-stride; cell I has
// linear index I_0 + N_0 (I_1 + N_1 I_2); face (I,i) is the LOWER face of cell I in direction i
// (coeff[I,i] multiplies p[I]-p[I-del(i)]).  L, u are n cell-sized fields back to
// back (component slowest).  The upper wall face I_i = N_i is not stored and has L = 0, u = 0.

#define _USE_MATH_DEFINES
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct Dims {
    int n;
    int64_t N[3];
    int64_t stride[3];
    int64_t M;
};

Dims make_dims(int n, const int64_t* d) {
    Dims g;
    g.n = n;
    for (int i = 0; i < 3; ++i) g.N[i] = (i < n) ? d[i] : 1;
    g.stride[0] = 1;
    g.stride[1] = g.N[0];
    g.stride[2] = g.N[0] * g.N[1];
    g.M = g.N[0] * g.N[1] * g.N[2];
    return g;
}

// ---------------------------------------------------------------------------------------------
// Operator.  BJ "Problem statement":
//   (A p)_I = sum_i [ L[I+di,i] (p[I+di] - p[I]) + L[I,i] (p[I-di] - p[I]) ],
// L = 0 on domain-boundary faces (Neumann); an out-of-range neighbour is never read.
// ---------------------------------------------------------------------------------------------
template <class T>
T apply_A_cell(const Dims& g, const T* L, const T* x, int64_t I0, int64_t I1, int64_t I2) {
    const int64_t Ii[3] = {I0, I1, I2};
    const int64_t I = I0 + g.N[0] * (I1 + g.N[1] * I2);
    T s = 0;
    for (int i = 0; i < g.n; ++i) {
        const T* Li = L + (int64_t)i * g.M;
        if (Ii[i] + 1 < g.N[i]) s += Li[I + g.stride[i]] * (x[I + g.stride[i]] - x[I]);
        if (Ii[i] > 0) s += Li[I] * (x[I - g.stride[i]] - x[I]);
    }
    return s;
}

// D_I = sum_i (L[I,i] + L[I+di,i]) = -diag(A)
template <class T>
T diag_cell(const Dims& g, const T* L, int64_t I0, int64_t I1, int64_t I2) {
    const int64_t Ii[3] = {I0, I1, I2};
    const int64_t I = I0 + g.N[0] * (I1 + g.N[1] * I2);
    T D = 0;
    for (int i = 0; i < g.n; ++i) {
        const T* Li = L + (int64_t)i * g.M;
        T Lm = (Ii[i] > 0) ? Li[I] : (T)0;
        T Lp = (Ii[i] + 1 < g.N[i]) ? Li[I + g.stride[i]] : (T)0;
        D += Lm + Lp;
    }
    return D;
}

template <class T>
void apply_A(const Dims& g, const T* L, const T* x, T* y) {
    for (int64_t I2 = 0; I2 < g.N[2]; ++I2)
        for (int64_t I1 = 0; I1 < g.N[1]; ++I1)
            for (int64_t I0 = 0; I0 < g.N[0]; ++I0)
                y[I0 + g.N[0] * (I1 + g.N[1] * I2)] = apply_A_cell(g, L, x, I0, I1, I2);
}

// r = b - A x
template <class T>
void residual(const Dims& g, const T* L, const T* x, const T* b, T* r) {
    for (int64_t I2 = 0; I2 < g.N[2]; ++I2)
        for (int64_t I1 = 0; I1 < g.N[1]; ++I1)
            for (int64_t I0 = 0; I0 < g.N[0]; ++I0) {
                int64_t I = I0 + g.N[0] * (I1 + g.N[1] * I2);
                r[I] = b[I] - apply_A_cell(g, L, x, I0, I1, I2);
            }
}

template <class T>
double max_abs(const T* v, int64_t M) {
    double m = 0;
    for (int64_t I = 0; I < M; ++I) {
        double a = std::fabs((double)v[I]);
        if (a > m) m = a;
    }
    return m;
}

// ---------------------------------------------------------------------------------------------
// Smoother.  BJ "Smoother: damped Jacobi, w = 2/3": every cell from the OLD x,
//   x_new = x + w invD (A x - b),  invD = D > 0 ? 1/D : 0   (diag(A) = -D; c-7, c-10).
// ---------------------------------------------------------------------------------------------
template <class T>
void jacobi_sweep(const Dims& g, const T* L, const T* x, const T* b, T* xnew) {
    const T omega = (T)(2.0 / 3.0);
    for (int64_t I2 = 0; I2 < g.N[2]; ++I2)
        for (int64_t I1 = 0; I1 < g.N[1]; ++I1)
            for (int64_t I0 = 0; I0 < g.N[0]; ++I0) {
                int64_t I = I0 + g.N[0] * (I1 + g.N[1] * I2);
                T D = diag_cell(g, L, I0, I1, I2);
                T invD = (D > (T)0) ? (T)1 / D : (T)0;
                T Ax = apply_A_cell(g, L, x, I0, I1, I2);
                xnew[I] = x[I] + omega * invD * (Ax - b[I]);
            }
}

template <class T>
void jacobi(const Dims& g, const T* L, T* x, const T* b, int sweeps, std::vector<T>& tmp) {
    tmp.resize((size_t)g.M);
    for (int s = 0; s < sweeps; ++s) {
        jacobi_sweep(g, L, x, b, tmp.data());
        std::memcpy(x, tmp.data(), sizeof(T) * (size_t)g.M);
    }
}

// ---------------------------------------------------------------------------------------------
// Transfers.  BJ "Restriction R sums the 2^n children; prolongation P is piecewise-constant
// injection"; "A coarse face coefficient is the sum of the 2^(n-1) fine face coefficients
// crossing it, so A_c = R·A·P exactly".
// ---------------------------------------------------------------------------------------------
template <class T>
void restrict_sum(const Dims& gf, const Dims& gc, const T* rf, T* rc) {
    for (int64_t J2 = 0; J2 < gc.N[2]; ++J2)
        for (int64_t J1 = 0; J1 < gc.N[1]; ++J1)
            for (int64_t J0 = 0; J0 < gc.N[0]; ++J0) {
                // children 2J + c, c in {0,1}^n; summed pairwise along axis 0, then 1, then 2 (c-12)
                T s2[2] = {0, 0};
                int n2 = (gf.n > 2) ? 2 : 1;
                for (int c2 = 0; c2 < n2; ++c2) {
                    T s1[2];
                    for (int c1 = 0; c1 < 2; ++c1) {
                        int64_t I = (2 * J0) + gf.N[0] * ((2 * J1 + c1) + gf.N[1] * ((gf.n > 2 ? 2 * J2 : 0) + c2));
                        s1[c1] = rf[I] + rf[I + 1];
                    }
                    s2[c2] = s1[0] + s1[1];
                }
                rc[J0 + gc.N[0] * (J1 + gc.N[1] * J2)] = (gf.n > 2) ? (s2[0] + s2[1]) : s2[0];
            }
}

template <class T>
void prolong_add(const Dims& gf, const Dims& gc, const T* xc, T* xf) {
    for (int64_t I2 = 0; I2 < gf.N[2]; ++I2)
        for (int64_t I1 = 0; I1 < gf.N[1]; ++I1)
            for (int64_t I0 = 0; I0 < gf.N[0]; ++I0) {
                int64_t J2 = (gf.n > 2) ? I2 / 2 : 0;
                xf[I0 + gf.N[0] * (I1 + gf.N[1] * I2)] += xc[(I0 / 2) + gc.N[0] * ((I1 / 2) + gc.N[1] * J2)];
            }
}

// Lc[i][J] = sum over the 2^(n-1) fine faces of direction i lying in coarse face (J,i):
// fine cells 2J + c with c_i = 0.  n = 3, tangential axes j < k: (c_j=0,c_k=0 + c_j=1,c_k=0) +
// (c_j=0,c_k=1 + c_j=1,c_k=1)  (fixed tree, c-12: the CUDA kernel must be bit-exact against this).
template <class T>
void coarsen(const Dims& gf, const Dims& gc, const T* Lf, T* Lc) {
    for (int i = 0; i < gf.n; ++i) {
        const T* Lfi = Lf + (int64_t)i * gf.M;
        T* Lci = Lc + (int64_t)i * gc.M;
        int tj = -1, tk = -1;  // tangential axes, ascending
        for (int a = 0; a < gf.n; ++a)
            if (a != i) { if (tj < 0) tj = a; else tk = a; }
        for (int64_t J2 = 0; J2 < gc.N[2]; ++J2)
            for (int64_t J1 = 0; J1 < gc.N[1]; ++J1)
                for (int64_t J0 = 0; J0 < gc.N[0]; ++J0) {
                    const int64_t J[3] = {J0, J1, J2};
                    int64_t base = 0;
                    for (int a = 0; a < gf.n; ++a) base += 2 * J[a] * gf.stride[a];
                    T s;
                    if (gf.n == 2) {
                        s = Lfi[base] + Lfi[base + gf.stride[tj]];
                    } else {
                        T a0 = Lfi[base] + Lfi[base + gf.stride[tj]];
                        T a1 = Lfi[base + gf.stride[tk]] + Lfi[base + gf.stride[tj] + gf.stride[tk]];
                        s = a0 + a1;
                    }
                    Lci[J0 + gc.N[0] * (J1 + gc.N[1] * J2)] = s;
                }
    }
}

// ---------------------------------------------------------------------------------------------
// H1 divergence: b[I] = sum_i (u[i][I+di] - u[i][I]); unstored upper wall face = 0.
// (BJ "Fused divergence"; configs[0] "b = sum_i (L u)[I+di,i] - (L u)[I,i]" with the masked
//  velocity passed in.)
// H8 gradient correction: u[i][I] -= L[i][I] (p[I] - p[I-di]); plane I_i = 0
// untouched (its L is 0 and p[I-di] does not exist).
// ---------------------------------------------------------------------------------------------
template <class T>
void divergence(const Dims& g, const T* u, T* b) {
    for (int64_t I2 = 0; I2 < g.N[2]; ++I2)
        for (int64_t I1 = 0; I1 < g.N[1]; ++I1)
            for (int64_t I0 = 0; I0 < g.N[0]; ++I0) {
                const int64_t Ii[3] = {I0, I1, I2};
                int64_t I = I0 + g.N[0] * (I1 + g.N[1] * I2);
                T s = 0;
                for (int i = 0; i < g.n; ++i) {
                    const T* ui = u + (int64_t)i * g.M;
                    T up = (Ii[i] + 1 < g.N[i]) ? ui[I + g.stride[i]] : (T)0;
                    s += up - ui[I];
                }
                b[I] = s;
            }
}

template <class T>
void gradient_correct(const Dims& g, const T* L, T* u, const T* p) {
    for (int i = 0; i < g.n; ++i) {
        const T* Li = L + (int64_t)i * g.M;
        T* ui = u + (int64_t)i * g.M;
        for (int64_t I2 = 0; I2 < g.N[2]; ++I2)
            for (int64_t I1 = 0; I1 < g.N[1]; ++I1)
                for (int64_t I0 = 0; I0 < g.N[0]; ++I0) {
                    const int64_t Ii[3] = {I0, I1, I2};
                    if (Ii[i] == 0) continue;
                    int64_t I = I0 + g.N[0] * (I1 + g.N[1] * I2);
                    ui[I] -= Li[I] * (p[I] - p[I - g.stride[i]]);
                }
    }
}

// ---------------------------------------------------------------------------------------------
// Hierarchy + V-cycle + solve + project (SURVEY.md §8(c) "Algorithm", each line from BJ).
// ---------------------------------------------------------------------------------------------
template <class T>
struct Level {
    Dims g;
    std::vector<T> L;  // n*M
    std::vector<T> x, b;  // levels >= 1 only
};

template <class T>
struct Ctx {
    int n;
    std::vector<Level<T>> lev;  // lev[0] = finest
    std::vector<T> tmp, r;
    bool have_coeff = false;
};

// BJ "The hierarchy halves every dimension down to a 4^n grid"; for general dims: coarsen while
// every extent is even and every half is >= 4 (c-4).
int num_coarsenings(int n, const int64_t* d) {
    int k = 0;
    int64_t N[3] = {d[0], d[1], n > 2 ? d[2] : 1};
    while (true) {
        bool ok = true;
        for (int i = 0; i < n; ++i)
            if (N[i] % 2 != 0 || N[i] / 2 < 4) ok = false;
        if (!ok) break;
        for (int i = 0; i < n; ++i) N[i] /= 2;
        ++k;
    }
    return k;
}

template <class T>
Ctx<T>* ctx_create(int n, const int64_t* d) {
    Ctx<T>* c = new Ctx<T>();
    c->n = n;
    int K = num_coarsenings(n, d);
    int64_t N[3] = {d[0], d[1], n > 2 ? d[2] : 1};
    for (int l = 0; l <= K; ++l) {
        Level<T> lv;
        lv.g = make_dims(n, N);
        lv.L.assign((size_t)(n * lv.g.M), (T)0);
        if (l > 0) {
            lv.x.assign((size_t)lv.g.M, (T)0);
            lv.b.assign((size_t)lv.g.M, (T)0);
        }
        c->lev.push_back(std::move(lv));
        for (int i = 0; i < n; ++i) N[i] /= 2;
    }
    return c;
}

// H0: level 0 = copy of the caller's L with the stored wall plane I_i = 0 forced to 0 (c-6); then
// one coarsening per level.
template <class T>
void ctx_set_coeff(Ctx<T>* c, const T* L) {
    Level<T>& f = c->lev[0];
    std::memcpy(f.L.data(), L, sizeof(T) * (size_t)(c->n * f.g.M));
    for (int i = 0; i < c->n; ++i)
        for (int64_t I2 = 0; I2 < f.g.N[2]; ++I2)
            for (int64_t I1 = 0; I1 < f.g.N[1]; ++I1)
                for (int64_t I0 = 0; I0 < f.g.N[0]; ++I0) {
                    const int64_t Ii[3] = {I0, I1, I2};
                    if (Ii[i] == 0) f.L[(size_t)(i * f.g.M + I0 + f.g.N[0] * (I1 + f.g.N[1] * I2))] = (T)0;
                }
    for (size_t l = 0; l + 1 < c->lev.size(); ++l)
        coarsen(c->lev[l].g, c->lev[l + 1].g, c->lev[l].L.data(), c->lev[l + 1].L.data());
    c->have_coeff = true;
}

// VCYCLE(l) on (x, b) of level l.
template <class T>
void vcycle(Ctx<T>* c, size_t l, T* x, const T* b) {
    Level<T>& lv = c->lev[l];
    const size_t last = c->lev.size() - 1;
    if (l == last) {
        // BJ "The coarsest level gets 64 Jacobi sweeps" (from x = 0 when it is a correction level;
        // with no coarsening at all the "cycle" is 64 sweeps from the current iterate)
        if (last > 0) std::fill(x, x + lv.g.M, (T)0);
        jacobi(lv.g, lv.L.data(), x, b, 64, c->tmp);
        return;
    }
    Level<T>& cv = c->lev[l + 1];
    jacobi(lv.g, lv.L.data(), x, b, 2, c->tmp);                        // BJ "2 pre-sweeps"
    std::vector<T> r((size_t)lv.g.M);
    residual(lv.g, lv.L.data(), x, b, r.data());                       // r = b - A x
    restrict_sum(lv.g, cv.g, r.data(), cv.b.data());                   // b_c = R r
    std::fill(cv.x.begin(), cv.x.end(), (T)0);                         // x_c = 0 (c-11)
    vcycle(c, l + 1, cv.x.data(), cv.b.data());
    prolong_add(lv.g, cv.g, cv.x.data(), x);                           // x += P x_c
    jacobi(lv.g, lv.L.data(), x, b, 2, c->tmp);                        // BJ "2 post-sweeps"
}

// p -= mean(p): sum in fp64 over all cells, subtract (T)mean (c-13).
template <class T>
void remove_mean(T* p, int64_t M) {
    double s = 0;
    for (int64_t I = 0; I < M; ++I) s += (double)p[I];
    T m = (T)(s / (double)M);
    for (int64_t I = 0; I < M; ++I) p[I] -= m;
}

template <class T>
double resnorm(Ctx<T>* c, const T* p, const T* b) {
    Level<T>& f = c->lev[0];
    c->r.resize((size_t)f.g.M);
    residual(f.g, f.L.data(), p, b, c->r.data());
    return max_abs(c->r.data(), f.g.M);
}

// One VCYCLE(0) + mean removal; returns ||b - A p||inf of the returned p.
template <class T>
double ctx_vcycle(Ctx<T>* c, T* p, const T* b) {
    vcycle(c, 0, p, b);
    remove_mean(p, c->lev[0].g.M);
    return resnorm(c, p, b);
}

// SOLVE (BJ "V-cycles repeat until ||r||inf <= 1e-4 ||b||inf or 32 cycles"): hist[0] before any
// cycle, hist[k] after k (c-14).  Returns 0 if converged, 1 if the cycle cap was reached.
template <class T>
int ctx_solve(Ctx<T>* c, T* p, const T* b, double tol, int maxcycles, double* hist, int* ncycles) {
    const int64_t M = c->lev[0].g.M;
    double nb = max_abs(b, M);
    hist[0] = resnorm(c, p, b);
    int k = 0;
    while (k < maxcycles && hist[k] > tol * nb) {
        hist[k + 1] = ctx_vcycle(c, p, b);
        ++k;
    }
    if (k == 0) remove_mean(p, M);
    *ncycles = k;
    return (hist[k] > tol * nb) ? 1 : 0;
}

// SOLVE_PCG — conjugate gradients on A p = b with ONE V-cycle (from a zero guess) as the
// preconditioner ("we now use Conjugate-Gradient smoothing within the GMG levels";
// reading 13 of DESIGN.md section 3: CG is wrapped around the multigrid cycle, the cycle itself —
// Jacobi sweeps, transfers, 64 coarse sweeps — stays the one of BJ).  A is negative semi-definite,
// the formulas are the textbook ones written with A itself (the two sign changes cancel):
//   r = b - A x;  hist[0] = ||r||inf
//   repeat while k < K and hist[k] > tol·||b||inf:
//     z = VCYCLE(0) applied to A z = r from z = 0;  mz = (T) mean(z)         (sum in fp64)
//     rho' = sum r_i z_i  (fp64, z before the shift);  beta = (T)(rho'/rho)  (first step: p = z - mz)
//     p = (z - mz) + beta p;  q = A p;  sigma = sum p_i q_i (fp64);  alpha = (T)(rho'/sigma)
//     x += alpha p;  r -= alpha q;  k++;  hist[k] = ||r||inf                  (recurrence residual)
//   x -= mean(x)
// Stops early (as converged) if rho' or sigma is exactly 0 (r = 0: nothing left to correct).
template <class T>
int ctx_solve_pcg(Ctx<T>* c, T* x, const T* b, double tol, int maxit, double* hist, int* nit) {
    Level<T>& f = c->lev[0];
    const int64_t M = f.g.M;
    std::vector<T> r((size_t)M), z((size_t)M), p((size_t)M, (T)0), q((size_t)M);
    const double nb = max_abs(b, M);
    residual(f.g, f.L.data(), x, b, r.data());
    hist[0] = max_abs(r.data(), M);
    double rho = 0;
    int k = 0;
    while (k < maxit && hist[k] > tol * nb) {
        std::fill(z.begin(), z.end(), (T)0);
        vcycle(c, 0, z.data(), r.data());                                 // z ~ A^-1 r
        double sz = 0, rho_new = 0;
        for (int64_t I = 0; I < M; ++I) { sz += (double)z[I]; rho_new += (double)r[I] * (double)z[I]; }
        const T mz = (T)(sz / (double)M);
        if (rho_new == 0.0) break;
        const T beta = (k == 0) ? (T)0 : (T)(rho_new / rho);
        for (int64_t I = 0; I < M; ++I) {
            const T zs = z[I] - mz;
            const T bp = beta * p[I];
            p[I] = zs + bp;
        }
        rho = rho_new;
        apply_A(f.g, f.L.data(), p.data(), q.data());
        double sigma = 0;
        for (int64_t I = 0; I < M; ++I) sigma += (double)p[I] * (double)q[I];
        if (sigma == 0.0) break;
        const T alpha = (T)(rho / sigma);
        for (int64_t I = 0; I < M; ++I) {
            const T ap = alpha * p[I];
            x[I] = x[I] + ap;
            const T aq = alpha * q[I];
            r[I] = r[I] - aq;
        }
        ++k;
        hist[k] = max_abs(r.data(), M);
    }
    remove_mean(x, M);
    *nit = k;
    return (hist[k] > tol * nb) ? 1 : 0;
}

// PROJECT (PAPER.md:29-33 + BJ "wl_project(u, L, p), which computes the divergence, solves, and
// corrects u").
template <class T>
int ctx_project(Ctx<T>* c, T* u, const T* L, T* p, double tol, int maxcycles, double* hist, int* ncycles) {
    if (L) ctx_set_coeff(c, L);
    Level<T>& f = c->lev[0];
    std::vector<T> b((size_t)f.g.M);
    divergence(f.g, u, b.data());
    int rc = ctx_solve(c, p, b.data(), tol, maxcycles, hist, ncycles);
    gradient_correct(f.g, f.L.data(), u, p);
    return rc;
}

// ---------------------------------------------------------------------------------------------
// BDIM coefficients from analytic bodies (NEXT-3).  BJ "BDIM face coefficient L = mu0(d): 0 for
// d <= -1, 1 for d >= 1, otherwise 0.5(1 + d + sin(pi d)/pi), where d is the signed distance to the
// body in cells, taken at the face centre and positive in the fluid."  Several bodies: d = min.
// Evaluated in fp64, clamped to [0,1], then cast (c-8); face (I,i) has coordinate I_i along i and
// I_j + 1/2 along the other axes (c-9); the stored wall plane I_i = 0 is 0 (c-6).
// Body record (8 doubles): kind (0 sphere / circle, 1 torus about axis 0), c0, c1, c2, R, r, -, -.
// ---------------------------------------------------------------------------------------------
double mu0(double d) {
    if (d <= -1.0) return 0.0;
    if (d >= 1.0) return 1.0;
    double v = 0.5 * (1.0 + d + std::sin(M_PI * d) / M_PI);
    if (v < 0.0) v = 0.0;
    if (v > 1.0) v = 1.0;
    return v;
}

double body_distance(int n, const double* B, const double* x) {
    const double dx = x[0] - B[1], dy = x[1] - B[2], dz = (n > 2) ? x[2] - B[3] : 0.0;
    if ((int)B[0] == 0) {
        double r2 = dx * dx + dy * dy;
        if (n > 2) r2 = r2 + dz * dz;
        return std::sqrt(r2) - B[4];
    }
    const double rho = std::sqrt(dy * dy + dz * dz) - B[4];
    return std::sqrt(rho * rho + dx * dx) - B[5];
}

template <class T>
void body_coeff(const Dims& g, int nbodies, const double* bodies, T* L) {
    for (int i = 0; i < g.n; ++i)
        for (int64_t I2 = 0; I2 < g.N[2]; ++I2)
            for (int64_t I1 = 0; I1 < g.N[1]; ++I1)
                for (int64_t I0 = 0; I0 < g.N[0]; ++I0) {
                    const int64_t Ii[3] = {I0, I1, I2};
                    const int64_t e = (int64_t)i * g.M + I0 + g.N[0] * (I1 + g.N[1] * I2);
                    if (Ii[i] == 0) { L[e] = (T)0; continue; }
                    double x[3];
                    for (int j = 0; j < 3; ++j) x[j] = (double)Ii[j] + ((j == i) ? 0.0 : 0.5);
                    double d = 1.0e300;
                    for (int k = 0; k < nbodies; ++k) {
                        const double dk = body_distance(g.n, bodies + 8 * k, x);
                        if (dk < d) d = dk;
                    }
                    L[e] = (T)mu0(d);
                }
}

// ---------------------------------------------------------------------------------------------
// CONVDIFF (the paper's `convdiff!` routine; "a third-order finite
// volume scheme ... implicit Large Eddy Simulation" PAPER.md:25).  The text gives the scheme's name only; every
// detail below is DESIGN.md section 3 reading 15:
//   r[i][I] = sum_j ( F_ij(I) - F_ij(I + d_j) )   for faces I_i >= 1,   r = 0 on the stored wall plane I_i = 0,
//   F_ij(I) = flux of u_i in direction j through the lower-j face of the control volume of u[i][I]
//           = U phi - nu (u[i][I] - u[i][I - d_j]),
//   U   = (u[j][I] + u[j][I - d_i]) / 2                       (advecting velocity, linear interpolation to the flux point)
//   phi = third-order upwind-biased face value of u_i along j: with C / D the values up / downstream of the flux point
//         (U >= 0: C = u[i][I-d_j], D = u[i][I], UU = u[i][I-2d_j];  U < 0: C = u[i][I], D = u[i][I-d_j], UU = u[i][I+d_j])
//         phi3 = (5 C + 2 D - UU) / 6   — the quadratic through three cell AVERAGES evaluated at the face (finite volume) —
//         limited to the monotone range (Leonard's universal limiter, constant slope 10):
//         phi = median(phi3, C, median(C, D, 10 C - 9 UU));  where UU lies outside the field, phi = (C + D) / 2.
//   Closed, impermeable, free-slip box (the Neumann walls of the projection, BJ "zero on domain-boundary faces"):
//   F_ij = 0 on the walls I_j = 0 and I_j = N_j for j != i; the unstored upper wall value u[i][N_i] is 0.
// Values are "defined" for 0 <= K_a <= N_a - 1 on every axis a != i and 0 <= K_i <= N_i.
// ---------------------------------------------------------------------------------------------
template <class T>
T median3(T a, T b, T c) {
    const T lo = (a < b) ? a : b;
    const T hi = (a < b) ? b : a;
    const T m = (hi < c) ? hi : c;
    return (lo < m) ? m : lo;
}

template <class T>
T face_value3(T uu, T c, T d) {
    const T phi3 = (T(5) * c + T(2) * d - uu) / T(6);
    const T bound = T(10) * c - T(9) * uu;
    return median3(phi3, c, median3(c, d, bound));
}

template <class T>
bool face_get(const Dims& g, const T* u, int i, const int64_t* K, T* v) {
    for (int a = 0; a < g.n; ++a) {
        if (K[a] < 0) return false;
        if (K[a] > ((a == i) ? g.N[a] : g.N[a] - 1)) return false;
    }
    if (K[i] == g.N[i]) { *v = (T)0; return true; }
    *v = u[(int64_t)i * g.M + K[0] + g.N[0] * (K[1] + g.N[1] * K[2])];
    return true;
}

template <class T>
T convdiff_flux(const Dims& g, const T* u, T nu, int i, int j, const int64_t* I) {
    if (j != i && (I[j] == 0 || I[j] == g.N[j])) return (T)0;
    int64_t K[3] = {I[0], I[1], I[2]};
    T a = 0, b = 0, p0 = 0, m1 = 0, uu = 0;
    face_get(g, u, j, K, &a);                 // u[j][I]
    K[i] -= 1; face_get(g, u, j, K, &b);      // u[j][I - d_i]
    K[i] += 1;
    const T U = T(0.5) * (a + b);
    face_get(g, u, i, K, &p0);                // u[i][I]
    K[j] -= 1; face_get(g, u, i, K, &m1);     // u[i][I - d_j]
    T C, D;
    bool have;
    if (U >= (T)0) { C = m1; D = p0; K[j] -= 1; have = face_get(g, u, i, K, &uu); }
    else { C = p0; D = m1; K[j] += 2; have = face_get(g, u, i, K, &uu); }
    const T phi = have ? face_value3(uu, C, D) : T(0.5) * (C + D);
    return U * phi - nu * (p0 - m1);
}

template <class T>
void convdiff(const Dims& g, const T* u, double nu_, T* r) {
    const T nu = (T)nu_;
    for (int i = 0; i < g.n; ++i)
        for (int64_t I2 = 0; I2 < g.N[2]; ++I2)
            for (int64_t I1 = 0; I1 < g.N[1]; ++I1)
                for (int64_t I0 = 0; I0 < g.N[0]; ++I0) {
                    const int64_t I[3] = {I0, I1, I2};
                    T s = 0;
                    if (I[i] > 0) {
                        for (int j = 0; j < g.n; ++j) {
                            int64_t Iu[3] = {I0, I1, I2};
                            Iu[j] += 1;
                            const T Fl = convdiff_flux(g, u, nu, i, j, I);
                            const T Fu = convdiff_flux(g, u, nu, i, j, Iu);
                            s = s + (Fl - Fu);
                        }
                    }
                    r[(int64_t)i * g.M + I0 + g.N[0] * (I1 + g.N[1] * I2)] = s;
                }
}

struct Handle {
    int dtype;  // 0 = f32, 1 = f64
    void* ctx;
};

}  // namespace

#define DISPATCH(h, expr_f, expr_d) \
    do { if ((h)->dtype == 0) { typedef float T; Ctx<T>* c = (Ctx<T>*)(h)->ctx; (void)c; expr_f; } \
         else { typedef double T; Ctx<T>* c = (Ctx<T>*)(h)->ctx; (void)c; expr_d; } } while (0)

extern "C" {

void* orc_create(int ndim, const int64_t* dims, int dtype) {
    if (ndim < 2 || ndim > 3 || (dtype != 0 && dtype != 1)) return nullptr;
    for (int i = 0; i < ndim; ++i) if (dims[i] < 4) return nullptr;
    Handle* h = new Handle();
    h->dtype = dtype;
    h->ctx = (dtype == 0) ? (void*)ctx_create<float>(ndim, dims) : (void*)ctx_create<double>(ndim, dims);
    return h;
}

void orc_destroy(void* hv) {
    Handle* h = (Handle*)hv;
    if (!h) return;
    if (h->dtype == 0) delete (Ctx<float>*)h->ctx; else delete (Ctx<double>*)h->ctx;
    delete h;
}

int orc_num_levels(void* hv) {
    Handle* h = (Handle*)hv;
    int r = 0;
    DISPATCH(h, r = (int)c->lev.size(), r = (int)c->lev.size());
    return r;
}

void orc_level_dims(void* hv, int level, int64_t* out) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, for (int i = 0; i < c->n; ++i) out[i] = c->lev[level].g.N[i],
                for (int i = 0; i < c->n; ++i) out[i] = c->lev[level].g.N[i]);
}

void orc_set_coeff(void* hv, const void* L) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, ctx_set_coeff(c, (const T*)L), ctx_set_coeff(c, (const T*)L));
}

void orc_get_coeff(void* hv, int level, void* out) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, std::memcpy(out, c->lev[level].L.data(), sizeof(T) * c->lev[level].L.size()),
                std::memcpy(out, c->lev[level].L.data(), sizeof(T) * c->lev[level].L.size()));
}

// y = A_level x
void orc_apply_A(void* hv, int level, const void* x, void* y) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, apply_A(c->lev[level].g, c->lev[level].L.data(), (const T*)x, (T*)y),
                apply_A(c->lev[level].g, c->lev[level].L.data(), (const T*)x, (T*)y));
}

// r = b - A_level x ; returns ||r||inf
double orc_residual(void* hv, int level, const void* x, const void* b, void* r) {
    Handle* h = (Handle*)hv;
    double m = 0;
    DISPATCH(h, (residual(c->lev[level].g, c->lev[level].L.data(), (const T*)x, (const T*)b, (T*)r),
                 m = max_abs((const T*)r, c->lev[level].g.M)),
                (residual(c->lev[level].g, c->lev[level].L.data(), (const T*)x, (const T*)b, (T*)r),
                 m = max_abs((const T*)r, c->lev[level].g.M)));
    return m;
}

// `sweeps` damped-Jacobi sweeps on level `level`, in place on x
void orc_jacobi(void* hv, int level, void* x, const void* b, int sweeps) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, jacobi(c->lev[level].g, c->lev[level].L.data(), (T*)x, (const T*)b, sweeps, c->tmp),
                jacobi(c->lev[level].g, c->lev[level].L.data(), (T*)x, (const T*)b, sweeps, c->tmp));
}

// rc = R r_f (level -> level+1)
void orc_restrict(void* hv, int level, const void* rf, void* rc) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, restrict_sum(c->lev[level].g, c->lev[level + 1].g, (const T*)rf, (T*)rc),
                restrict_sum(c->lev[level].g, c->lev[level + 1].g, (const T*)rf, (T*)rc));
}

// x_f += P x_c (level+1 -> level)
void orc_prolong_add(void* hv, int level, const void* xc, void* xf) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, prolong_add(c->lev[level].g, c->lev[level + 1].g, (const T*)xc, (T*)xf),
                prolong_add(c->lev[level].g, c->lev[level + 1].g, (const T*)xc, (T*)xf));
}

// VCYCLE(level) on caller arrays of that level (no mean removal)
void orc_vcycle_level(void* hv, int level, void* x, const void* b) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, vcycle(c, (size_t)level, (T*)x, (const T*)b), vcycle(c, (size_t)level, (T*)x, (const T*)b));
}

// one VCYCLE(0) + mean removal; returns ||b - A p||inf
double orc_vcycle(void* hv, void* p, const void* b) {
    Handle* h = (Handle*)hv;
    double r = 0;
    DISPATCH(h, r = ctx_vcycle(c, (T*)p, (const T*)b), r = ctx_vcycle(c, (T*)p, (const T*)b));
    return r;
}

int orc_solve(void* hv, void* p, const void* b, double tol, int maxcycles, double* hist, int* ncycles) {
    Handle* h = (Handle*)hv;
    int rc = 0;
    DISPATCH(h, rc = ctx_solve(c, (T*)p, (const T*)b, tol, maxcycles, hist, ncycles),
                rc = ctx_solve(c, (T*)p, (const T*)b, tol, maxcycles, hist, ncycles));
    return rc;
}

double orc_mu0(double d) { return mu0(d); }

// L (n*M elements of dtype) for `nbodies` bodies on a grid of `dims`
int orc_body_coeff(int ndim, const int64_t* dims, int dtype, int nbodies, const double* bodies, void* L) {
    if (ndim < 2 || ndim > 3) return -1;
    Dims g = make_dims(ndim, dims);
    if (dtype == 0) body_coeff(g, nbodies, bodies, (float*)L); else body_coeff(g, nbodies, bodies, (double*)L);
    return 0;
}

int orc_solve_pcg(void* hv, void* p, const void* b, double tol, int maxit, double* hist, int* nit) {
    Handle* h = (Handle*)hv;
    int rc = 0;
    DISPATCH(h, rc = ctx_solve_pcg(c, (T*)p, (const T*)b, tol, maxit, hist, nit),
                rc = ctx_solve_pcg(c, (T*)p, (const T*)b, tol, maxit, hist, nit));
    return rc;
}

int orc_project(void* hv, void* u, const void* L, void* p, double tol, int maxcycles, double* hist, int* ncycles) {
    Handle* h = (Handle*)hv;
    int rc = 0;
    DISPATCH(h, rc = ctx_project(c, (T*)u, (const T*)L, (T*)p, tol, maxcycles, hist, ncycles),
                rc = ctx_project(c, (T*)u, (const T*)L, (T*)p, tol, maxcycles, hist, ncycles));
    return rc;
}

void orc_divergence(void* hv, const void* u, void* b) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, divergence(c->lev[0].g, (const T*)u, (T*)b), divergence(c->lev[0].g, (const T*)u, (T*)b));
}

// u[i][I] -= L0[i][I] (p[I] - p[I-di]) with the ctx's level-0 coefficients
void orc_gradient_correct(void* hv, void* u, const void* p) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, gradient_correct(c->lev[0].g, c->lev[0].L.data(), (T*)u, (const T*)p),
                gradient_correct(c->lev[0].g, c->lev[0].L.data(), (T*)u, (const T*)p));
}

// p -= mean(p)
void orc_remove_mean(void* hv, void* p) {
    Handle* h = (Handle*)hv;
    DISPATCH(h, remove_mean((T*)p, c->lev[0].g.M), remove_mean((T*)p, c->lev[0].g.M));
}

// NEXT-4: r = convdiff(u; nu) on a grid of `dims` (no context needed).  dtype 0 = f32, 1 = f64.
int orc_convdiff(int ndim, const int64_t* dims, int dtype, const void* u, double nu, void* r) {
    if (ndim < 2 || ndim > 3) return -1;
    const Dims g = make_dims(ndim, dims);
    if (dtype == 0) convdiff<float>(g, (const float*)u, nu, (float*)r);
    else convdiff<double>(g, (const double*)u, nu, (double*)r);
    return 0;
}
// the limited third-order face value of (UU, C, D), in the given precision (returned as double)
double orc_face_value(int dtype, double uu, double c, double d) {
    if (dtype == 0) return (double)face_value3<float>((float)uu, (float)c, (float)d);
    return face_value3<double>(uu, c, d);
}

}  // extern "C"
