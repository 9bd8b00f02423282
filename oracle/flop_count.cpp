// flop_count.cpp -- TEST INFRASTRUCTURE.  Counts the floating-point operations of the oracle's own formulas
// (oracle/hydro_oracle.cpp, included verbatim below) by instantiating them on a counting scalar type, and
// assembles from the pieces the ALGORITHMIC flops per cell of one L(u) and of one RK3 step under the convention
// of SURVEY.md section 8(d) / DESIGN.md section 8:
//     add, sub, mul, div, sqrt, abs, max, min = 1 flop each; comparisons and sign flips = 0;
//     per cell: con2prim once, the three signal speeds once, the physical flux once per direction;
//     per interface and direction: the alpha max, the split of the 2(2r-1) stencil values of each field,
//     ten reconstructions, five sums; per cell and direction the divergence; per step the RK combination.
// (The oracle itself recomputes the physical flux and the speed of every stencil cell at every interface; that
// redundancy is not algorithmic and is not counted: the pieces are counted one by one.)
//
// Build and run:  g++ -O1 -std=c++17 oracle/flop_count.cpp -o /tmp/flop_count && /tmp/flop_count
// oracle/flop_count.py does that and checks bench.py's constants (tests/test_flop_count.py).
#include <cmath>
#include <cstdio>

struct Counted {
    double v;
    static long long n_add, n_mul, n_div, n_sqrt, n_minmax;
    Counted() : v(0) {}
    Counted(double x) : v(x) {}
    Counted(int x) : v(x) {}
    explicit operator double() const { return v; }
    static void reset() { n_add = n_mul = n_div = n_sqrt = n_minmax = 0; }
    static long long total() { return n_add + n_mul + n_div + n_sqrt + n_minmax; }
};
long long Counted::n_add = 0, Counted::n_mul = 0, Counted::n_div = 0, Counted::n_sqrt = 0, Counted::n_minmax = 0;

inline Counted operator+(Counted a, Counted b) { ++Counted::n_add; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { ++Counted::n_add; return Counted(a.v - b.v); }
inline Counted operator*(Counted a, Counted b) { ++Counted::n_mul; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { ++Counted::n_div; return Counted(a.v / b.v); }
inline Counted operator-(Counted a) { return Counted(-a.v); }
inline Counted& operator+=(Counted& a, Counted b) { a = a + b; return a; }
inline Counted& operator*=(Counted& a, Counted b) { a = a * b; return a; }
inline bool operator<(Counted a, Counted b) { return a.v < b.v; }
inline bool operator>(Counted a, Counted b) { return a.v > b.v; }
inline bool operator<=(Counted a, Counted b) { return a.v <= b.v; }
inline bool operator>=(Counted a, Counted b) { return a.v >= b.v; }
// mixed forms the oracle's templates use (int and double literals)
inline Counted operator*(int a, Counted b) { return Counted(a) * b; }
inline Counted operator*(Counted a, int b) { return a * Counted(b); }
inline Counted operator*(double a, Counted b) { return Counted(a) * b; }
inline Counted operator-(int a, Counted b) { return Counted(a) - b; }
inline bool operator>(Counted a, int b) { return a.v > b; }

namespace std {   // the oracle calls these qualified; declared before its templates are parsed
inline Counted sqrt(Counted a) { ++Counted::n_sqrt; return Counted(std::sqrt(a.v)); }
inline Counted fabs(Counted a) { ++Counted::n_minmax; return Counted(std::fabs(a.v)); }
inline Counted fmax(Counted a, Counted b) { ++Counted::n_minmax; return Counted(std::fmax(a.v, b.v)); }
inline Counted fmin(Counted a, Counted b) { ++Counted::n_minmax; return Counted(std::fmin(a.v, b.v)); }
}  // namespace std

#include "hydro_oracle.cpp"

namespace {

long long count_con2prim() {
    Counted u[NF] = {2.0, 0.3, -0.2, 0.1, 0.7};
    int flag = 0;
    Counted::reset();
    (void)con2prim<Counted>(u, &flag);
    return Counted::total();
}
long long count_speed() {
    Counted v[3] = {0.2, -0.1, 0.3};
    Counted::reset();
    (void)signal_speed<Counted>(v, 0);
    return Counted::total();
}
long long count_phys_flux() {
    Counted u[NF] = {2.0, 0.3, -0.2, 0.1, 0.7};
    int flag = 0;
    const Prim<Counted> w = con2prim<Counted>(u, &flag);
    Counted F[NF];
    Counted::reset();
    phys_flux<Counted>(u, w, 0, F);
    return Counted::total();   // the "+ 0" of the off-diagonal pressure terms is counted by the type: see main()
}
long long count_weno(int r) {
    Counted f[7] = {1.0, 1.2, 1.1, 1.5, 1.4, 1.45, 1.3};
    Counted::reset();
    if (r == 3) (void)weno5<Counted>(f, Counted(1e-6));
    else (void)weno7<Counted>(f, Counted(1e-6));
    return Counted::total();
}
// alpha max + split + reconstructions + sums of one interface and direction, physical flux and speeds given
long long count_llf_split(int r) {
    Counted cells[8][NF], F[8][NF], a[8], fh[NF];
    for (int k = 0; k < 8; ++k) {
        a[k] = Counted(0.5 + 0.01 * k);
        for (int c = 0; c < NF; ++c) { cells[k][c] = Counted(1.0 + 0.1 * k + c); F[k][c] = Counted(0.5 + 0.07 * k - c); }
    }
    Counted::reset();
    llf_weno_split<Counted>(r, cells, F, a, Counted(1e-6), fh);
    return Counted::total();
}
long long count_musta(int K) {
    Counted cells[4][NF];
    for (int k = 0; k < 4; ++k) {
        cells[k][0] = Counted(2.0 + 0.1 * k);
        cells[k][1] = Counted(0.3 + 0.02 * k); cells[k][2] = Counted(-0.2 + 0.01 * k); cells[k][3] = Counted(0.1);
        cells[k][4] = Counted(0.7 + 0.03 * k);
    }
    Counted fs[NF];
    int flag = 0;
    Counted::reset();
    musta_force_flux<Counted>(cells, 0, K, Counted(0.9), fs, &flag);
    return Counted::total();
}

}  // namespace

int main() {
    const long long c2p = count_con2prim(), spd = count_speed();
    // phys_flux adds "p or 0" to each of the three momentum fluxes; only the one real addition is algorithmic
    const long long flx = count_phys_flux() - 2;
    const long long w5 = count_weno(3), w7 = count_weno(4);
    const long long s5 = count_llf_split(3), s7 = count_llf_split(4);
    const long long mu = count_musta(2);
    const long long div = 2 * NF;                 // (f_lo - f_hi) / dx per field and direction
    const long long rk = 4 * NF + 4 * NF + 2 * NF;  // stage 2 and 3: 4 ops per field, stage 1: 2
    const long long L5 = c2p + 3 * spd + 3 * (flx + s5 + div);
    const long long L7 = c2p + 3 * spd + 3 * (flx + s7 + div);
    const long long LM = 3 * (mu + div);
    printf("con2prim %lld\nsignal_speed %lld\nphys_flux %lld\nweno5 %lld\nweno7 %lld\n", c2p, spd, flx, w5, w7);
    printf("llf_split_weno5 %lld\nllf_split_weno7 %lld\nmusta_force_K2 %lld\n", s5, s7, mu);
    printf("L_weno5 %lld\nL_weno7 %lld\nL_musta %lld\n", L5, L7, LM);
    printf("step_weno5 %lld\nstep_weno7 %lld\nstep_musta %lld\n", 3 * L5 + rk, 3 * L7 + rk, 3 * LM + rk);
    return 0;
}
