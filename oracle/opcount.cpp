// oracle/opcount.cpp -- TEST/MEASUREMENT INFRASTRUCTURE (see mhd_oracle.h).
// Counts the floating-point operations the oracle performs, by compiling the very same
// source (mhd_oracle.c) with `real` replaced by a counting type.  Used to state the
// ALGORITHMIC flops per cell-update in DESIGN.md / bench.py's roofline; it is not part
// of the product path.   g++ -O1 -std=c++17 oracle/opcount.cpp -o oracle/opcount && oracle/opcount [n [2d]]
// ("2d": patches of n x n x 1 cells, z collapsed -- the count behind the 2D tile kernel's roofline)
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

struct Ops { long long add, mul, div, sqrt_, cmp, minmaxabs; };
static Ops g = {0, 0, 0, 0, 0, 0};

struct Counted {
  double v;
  Counted() : v(0) {}
  Counted(double x) : v(x) {}
  Counted(int x) : v(x) {}
  explicit operator double() const { return v; }
};
static inline Counted operator+(Counted a, Counted b) { ++g.add; return Counted(a.v + b.v); }
static inline Counted operator-(Counted a, Counted b) { ++g.add; return Counted(a.v - b.v); }
static inline Counted operator*(Counted a, Counted b) { ++g.mul; return Counted(a.v * b.v); }
static inline Counted operator/(Counted a, Counted b) { ++g.div; return Counted(a.v / b.v); }
static inline Counted operator-(Counted a) { return Counted(-a.v); }
static inline Counted& operator+=(Counted& a, Counted b) { a = a + b; return a; }
static inline Counted& operator-=(Counted& a, Counted b) { a = a - b; return a; }
static inline bool operator<(Counted a, Counted b) { ++g.cmp; return a.v < b.v; }
static inline bool operator>(Counted a, Counted b) { ++g.cmp; return a.v > b.v; }
static inline bool operator<=(Counted a, Counted b) { ++g.cmp; return a.v <= b.v; }
static inline bool operator>=(Counted a, Counted b) { ++g.cmp; return a.v >= b.v; }
static inline bool operator==(Counted a, Counted b) { ++g.cmp; return a.v == b.v; }
static inline Counted sqrt(Counted a) { ++g.sqrt_; return Counted(std::sqrt(a.v)); }
static inline Counted fabs(Counted a) { ++g.minmaxabs; return Counted(std::fabs(a.v)); }

#define ORACLE_REAL Counted
extern "C++" {
#include "mhd_oracle.c"
}

static Ops snap() { return g; }
static Ops diff(Ops a, Ops b) { return {a.add - b.add, a.mul - b.mul, a.div - b.div, a.sqrt_ - b.sqrt_, a.cmp - b.cmp, a.minmaxabs - b.minmaxabs}; }
static void show(const char* name, Ops o, double per) {
  std::printf("%-34s add %8.1f mul %8.1f div %7.1f sqrt %6.1f | flops %8.1f | cmp %7.1f abs %6.1f\n", name, o.add / per,
              o.mul / per, o.div / per, o.sqrt_ / per, (o.add + o.mul + o.div + o.sqrt_) / per, o.cmp / per, o.minmaxabs / per);
}

int main(int argc, char** argv) {
  const int n = argc > 1 ? std::atoi(argv[1]) : 32;
  const bool two_d = argc > 2 && std::strcmp(argv[2], "2d") == 0;
  // a smooth, fully three-dimensional state on 2 patches of n^3 (values only matter
  // for which HLLD branch is taken; the count per call is branch-independent up to selects)
  orc_desc d;
  std::memset(&d, 0, sizeof d);
  d.n[0] = d.n[1] = d.n[2] = n; d.ng = 3; d.npatch = 2; d.limiter = 1; d.emf_solver = 0;
  if (two_d) d.n[2] = 1;
  d.gamma = 5.0 / 3.0; d.dx[0] = d.dx[1] = d.dx[2] = 1.0 / (2 * n);
  const long m = n + 6, M = m * m * (two_d ? 1 : m);
  std::vector<Counted> U(8 * 2 * M), V(8 * 2 * M);
  for (int f = 0; f < 8; ++f)
    for (long c = 0; c < 2 * M; ++c) {
      const double x = 0.37 * (c % m) + 0.11 * ((c / m) % m) + 0.05 * (c / (m * m));
      const double base[8] = {1.0, 0.3, -0.2, 0.1, 3.0, 0.1, 0.05, -0.07};
      U[f * 2 * M + c] = base[f] * (1.0 + 0.1 * std::sin(x + f));
    }
  const double cells = 2.0 * n * n * (two_d ? 1 : n);
  Ops a = snap();
  orc_step(&d, U.data(), V.data(), 1e-3);
  Ops b = snap();
  show("whole step, per interior cell", diff(b, a), cells);
  a = snap();
  double dt = orc_cfl_dt(&d, U.data(), 0.4, nullptr);
  b = snap();
  show("cfl_dt, per interior cell", diff(b, a), cells);
  (void)dt;
  // pointwise solvers
  Counted L[7] = {1.0, 0.3, 0.1, -0.2, 1.0, 0.5, 0.2}, R[7] = {0.8, -0.1, 0.2, 0.1, 0.7, 0.4, -0.3}, F[7];
  a = snap();
  orc_hlld(5.0 / 3.0, L, R, Counted(0.6), F);
  b = snap();
  show("one HLLD solve (7 fluxes)", diff(b, a), 1.0);
  Counted c4[4][6] = {{1.0, 0.3, 0.1, -0.2, 1.0, 0.5}, {0.9, 0.2, -0.1, 0.1, 0.8, 0.4}, {1.1, 0.1, 0.2, 0.0, 1.2, 0.3}, {0.8, -0.2, 0.1, 0.3, 0.9, 0.2}};
  a = snap();
  Counted e = orc_emf2d(5.0 / 3.0, 0, c4, Counted(0.3), Counted(0.35), Counted(-0.2), Counted(-0.25));
  b = snap();
  show("one HLLD-2D edge solve", diff(b, a), 1.0);
  a = snap();
  e = orc_emf2d(5.0 / 3.0, 1, c4, Counted(0.3), Counted(0.35), Counted(-0.2), Counted(-0.25));
  b = snap();
  show("one HLL-2D edge solve", diff(b, a), 1.0);
  (void)e;
  return 0;
}
