// fx_compiler.cpp -- host compiler of the integrand texts.
//
// Pipeline:
//   1. parse the worker grammar into a hash-consed DAG shared by the K
//      orders of a sector, so identical f-lines are evaluated once per point (R7);
//   2. lower: every additive/multiplicative region becomes a sparse polynomial over "atoms"
//      (variables, or opaque sub-results such as log F, U^p, a quotient).  Sums are only
//      re-associated and monomial x polynomial products distributed; polynomial x polynomial is
//      never expanded, so no cancellation is introduced (R14);
//      p[e,q] with non-integer q becomes exp(q*log e) and shares log e with l[e] (R9);
//   3. emit accumulator-machine code (fx_isa.h): greedy multivariate Horner for the
//      polynomials (one FMA per factoring step), register temporaries S[0..7] allocated by
//      liveness, overflow to shared-memory slots M[];
//   4. for contour deformation (R11): expand F fully, differentiate the monomial
//      list symbolically once and twice, emit a real program that leaves dF/dx_k and
//      d2F/dx_k dx_l in M[].
#include "fx_compiler.hpp"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <set>
#include <tuple>

namespace fx {
namespace {

#ifndef FX_HORNER_LOOK
#define FX_HORNER_LOOK 1
#endif
#ifndef FX_HORNER_CAND
#define FX_HORNER_CAND 4
#endif

[[noreturn]] void fail(int code, const std::string &msg) { throw CompileError{code, msg}; }

// ------------------------------------------------------------------------------ raw DAG
enum RK : uint8_t { R_CONST, R_VAR, R_ADD, R_SUB, R_MUL, R_DIV, R_NEG, R_POWI, R_POWR, R_LOG };

struct RNode {
  RK k;
  int a = -1, b = -1;
  double c = 0.0;  // constant value, or real exponent
  int n = 0;       // variable index (0-based), or integer exponent
};

uint64_t dbits(double d) {
  uint64_t u;
  std::memcpy(&u, &d, 8);
  return u;
}

struct RawDag {
  std::vector<RNode> nodes;
  std::map<std::tuple<int, int, int, uint64_t, int>, int> index;
  int make(RK k, int a, int b, double c, int n) {
    auto key = std::make_tuple((int)k, a, b, dbits(c), n);
    auto it = index.find(key);
    if (it != index.end()) return it->second;
    nodes.push_back(RNode{k, a, b, c, n});
    index.emplace(key, (int)nodes.size() - 1);
    return (int)nodes.size() - 1;
  }
};

// psi^(n)(m) = (-1)^(n+1) n! (zeta(n+1) - sum_{j<m} j^-(n+1)) for the pairs of PAPER.md:515.
double polygamma_const(int n, int m) {
  const long double pi = 3.14159265358979323846264338327950288L;
  const long double zeta3 = 1.20205690315959428539973816151144999L;
  long double z;
  if (n == 1) z = pi * pi / 6.0L;
  else if (n == 2) z = zeta3;
  else z = pi * pi * pi * pi / 90.0L;
  long double tail = 0.0L;
  for (int j = 1; j < m; ++j) tail += 1.0L / powl((long double)j, n + 1);
  long double fact = 1.0L;
  for (int j = 2; j <= n; ++j) fact *= j;
  long double sign = ((n + 1) % 2 == 0) ? 1.0L : -1.0L;
  return (double)(sign * fact * (z - tail));
}

// ------------------------------------------------------------------------------ parser
struct Parser {
  RawDag &dag;
  const std::string &s;
  size_t pos;
  int nvars;
  const std::vector<int> &funcs;  // ids of f[1..] defined so far
  std::set<int> &fbound;
  std::string where;

  [[noreturn]] void err(const std::string &m) {
    fail(FIESTA_E_PARSE, where + ": " + m + " at column " + std::to_string(pos + 1) + " of '" +
                             (s.size() > 60 ? s.substr(0, 60) + "..." : s) + "'");
  }
  void ws() {
    while (pos < s.size() && std::isspace((unsigned char)s[pos])) ++pos;
  }
  bool peek(char c) {
    ws();
    return pos < s.size() && s[pos] == c;
  }
  bool eat(char c) {
    if (peek(c)) {
      ++pos;
      return true;
    }
    return false;
  }
  void need(char c) {
    if (!eat(c)) err(std::string("expected '") + c + "'");
  }
  bool number(double &out, bool &is_int, long &ival) {
    ws();
    size_t p = pos;
    size_t d0 = p;
    while (p < s.size() && std::isdigit((unsigned char)s[p])) ++p;
    bool intdigits = p > d0;
    bool dot = false;
    size_t fracdigits = 0;
    if (p < s.size() && s[p] == '.') {
      dot = true;
      ++p;
      size_t f0 = p;
      while (p < s.size() && std::isdigit((unsigned char)s[p])) ++p;
      fracdigits = p - f0;
    }
    if (!intdigits && fracdigits == 0) return false;
    bool hasexp = false;
    if (p < s.size() && (s[p] == 'e' || s[p] == 'E')) {
      size_t q = p + 1;
      if (q < s.size() && (s[q] == '+' || s[q] == '-')) ++q;
      size_t e0 = q;
      while (q < s.size() && std::isdigit((unsigned char)s[q])) ++q;
      if (q > e0) {
        p = q;
        hasexp = true;
      }
    }
    std::string tok = s.substr(pos, p - pos);
    out = std::strtod(tok.c_str(), nullptr);  // nearest FP64 value of the literal ("doubles")
    is_int = intdigits && !dot && !hasexp;
    ival = is_int ? std::strtol(tok.c_str(), nullptr, 10) : 0;
    pos = p;
    return true;
  }
  int index_in_brackets() {
    need('[');
    double v;
    bool is_int;
    long iv;
    if (!number(v, is_int, iv) || !is_int) err("index must be a positive integer");
    need(']');
    return (int)iv;
  }
  double signed_number() {
    double sign = 1.0;
    for (;;) {
      if (eat('-')) sign = -sign;
      else if (eat('+')) {
      } else break;
    }
    double v;
    bool is_int;
    long iv;
    if (!number(v, is_int, iv)) err("expected a number");
    return sign * v;
  }
  int expr() {
    int a = term();
    for (;;) {
      if (eat('+')) a = dag.make(R_ADD, a, term(), 0, 0);
      else if (eat('-')) a = dag.make(R_SUB, a, term(), 0, 0);
      else return a;
    }
  }
  int term() {
    int a = unary();
    for (;;) {
      if (eat('*')) a = dag.make(R_MUL, a, unary(), 0, 0);
      else if (eat('/')) a = dag.make(R_DIV, a, unary(), 0, 0);
      else return a;
    }
  }
  int unary() {
    if (eat('-')) return dag.make(R_NEG, unary(), -1, 0, 0);
    if (eat('+')) return unary();
    return atom();
  }
  bool word(const char *w) {
    ws();
    size_t n = std::strlen(w);
    if (s.compare(pos, n, w) == 0) {
      pos += n;
      return true;
    }
    return false;
  }
  int atom() {
    ws();
    double v;
    bool is_int;
    long iv;
    if (number(v, is_int, iv)) return dag.make(R_CONST, -1, -1, v, 0);
    if (eat('(')) {
      int e = expr();
      need(')');
      return e;
    }
    if (word("PolyGamma")) {
      need('[');
      double a, b;
      bool ai, bi;
      long an, bn;
      if (!number(a, ai, an) || !ai) err("PolyGamma arguments must be integers");
      need(',');
      if (!number(b, bi, bn) || !bi) err("PolyGamma arguments must be integers");
      need(']');
      static const int ok[7][2] = {{1, 1}, {2, 1}, {2, 2}, {2, 3}, {2, 4}, {3, 1}, {3, 2}};
      for (auto &p : ok)
        if (p[0] == an && p[1] == bn) return dag.make(R_CONST, -1, -1, polygamma_const((int)an, (int)bn), 0);
      err("PolyGamma[" + std::to_string(an) + "," + std::to_string(bn) + "] is not hard-coded (PAPER.md:515)");
    }
    if (pos < s.size()) {
      char c = s[pos];
      if (c == 'x') {
        ++pos;
        int i = index_in_brackets();
        if (i < 1 || i > nvars) fail(FIESTA_E_DIM, where + ": x[" + std::to_string(i) + "] out of range 1.." + std::to_string(nvars));
        return dag.make(R_VAR, -1, -1, 0, i - 1);
      }
      if (c == 'f') {
        ++pos;
        int i = index_in_brackets();
        if (i < 1 || i > (int)funcs.size()) err("f[" + std::to_string(i) + "] used before it is defined");
        fbound.insert(funcs[i - 1]);
        return funcs[i - 1];
      }
      if (c == 'p') {
        ++pos;
        need('[');
        int e = expr();
        need(',');
        bool paren = eat('(');
        double q = signed_number();
        if (eat('/')) q = q / signed_number();
        if (paren) need(')');
        need(']');
        if (q == std::floor(q) && std::fabs(q) < 1e6) return dag.make(R_POWI, e, -1, 0, (int)q);
        return dag.make(R_POWR, e, -1, q, 0);
      }
      if (c == 'l') {
        ++pos;
        need('[');
        int e = expr();
        need(']');
        return dag.make(R_LOG, e, -1, 0, 0);
      }
      if (c == 'P') {
        ++pos;
        return dag.make(R_CONST, -1, -1, 3.14159265358979323846, 0);
      }
      if (c == 'G') {
        ++pos;
        return dag.make(R_CONST, -1, -1, 0.57721566490153286061, 0);
      }
    }
    err("unexpected input");
  }
};

int parse_line(RawDag &dag, const std::string &line, int nvars, const std::vector<int> &funcs, std::set<int> &fbound,
               const std::string &where) {
  Parser p{dag, line, 0, nvars, funcs, fbound, where};
  int e = p.expr();
  p.ws();
  if (p.pos != line.size()) p.err("trailing input after expression");
  return e;
}

std::string trim(const std::string &s) {
  size_t a = 0, b = s.size();
  while (a < b && std::isspace((unsigned char)s[a])) ++a;
  while (b > a && std::isspace((unsigned char)s[b - 1])) --b;
  return s.substr(a, b - a);
}

bool all_digits(const std::string &s) {
  if (s.empty()) return false;
  for (char c : s)
    if (!std::isdigit((unsigned char)c)) return false;
  return true;
}

// One block "<nvars>; <nfuncs>; f1; ...; final; |"  ->  ids of the f-lines and of the final expression.
void parse_block(RawDag &dag, const char *text, int dim, std::set<int> &fbound, const std::string &where,
                 std::vector<int> &funcs, int &final_id) {
  std::string body(text);
  size_t bar = body.find('|');
  if (bar != std::string::npos) {
    if (!trim(body.substr(bar + 1)).empty()) fail(FIESTA_E_PARSE, where + ": text after the terminating '|'");
    body = body.substr(0, bar);
  }
  std::vector<std::string> fields;
  size_t start = 0;
  for (;;) {
    size_t sc = body.find(';', start);
    if (sc == std::string::npos) {
      fields.push_back(body.substr(start));
      break;
    }
    fields.push_back(body.substr(start, sc - start));
    start = sc + 1;
  }
  if (!trim(fields.back()).empty()) fail(FIESTA_E_PARSE, where + ": every expression line must end with ';'");
  fields.pop_back();
  for (auto &f : fields) f = trim(f);
  if (fields.size() < 3) fail(FIESTA_E_PARSE, where + ": need number of variables; number of functions; final expression;");
  if (!all_digits(fields[0]) || !all_digits(fields[1]))
    fail(FIESTA_E_PARSE, where + ": the first two lines must be non-negative integers");
  int nvars = std::atoi(fields[0].c_str()), nf = std::atoi(fields[1].c_str());
  if (nvars != dim) fail(FIESTA_E_DIM, where + ": text declares " + std::to_string(nvars) + " variables, dim is " + std::to_string(dim));
  if ((int)fields.size() != 2 + nf + 1)
    fail(FIESTA_E_PARSE, where + ": expected " + std::to_string(nf) + " function lines and one final expression, got " +
                             std::to_string(fields.size() - 2) + " lines");
  funcs.clear();
  for (int k = 0; k < nf; ++k)
    funcs.push_back(parse_line(dag, fields[2 + k], nvars, funcs, fbound, where + " f[" + std::to_string(k + 1) + "]"));
  final_id = parse_line(dag, fields[2 + nf], nvars, funcs, fbound, where + " final");
}

// ------------------------------------------------------------------------------ lowering
struct Term {
  double c;
  std::vector<std::pair<int, int>> f;  // (atom id, exponent >= 1), sorted by atom id
};
typedef std::vector<Term> Poly;

enum LK : uint8_t { L_VAR, L_CONST, L_POLY, L_DIV, L_LOG, L_EXP, L_POWI, L_SQRT };

struct Opnd {
  enum Kind { NONE, IMM, REG, MEM } kind = NONE;
  int idx = 0;
  double c = 0.0;
};

struct LNode {
  LK k;
  int a = -1, b = -1;
  double c = 0.0;
  int n = 0;
  Poly terms;
  int uses = 0, rem = 0;
  bool mat = false;
  Opnd loc;
};

void normalize(Poly &p) {
  std::sort(p.begin(), p.end(), [](const Term &x, const Term &y) { return x.f < y.f; });
  Poly out;
  for (auto &t : p) {
    if (!out.empty() && out.back().f == t.f) out.back().c += t.c;
    else out.push_back(t);
  }
  Poly out2;
  for (auto &t : out)
    if (t.c != 0.0) out2.push_back(t);
  p.swap(out2);
}

Term mul_terms(const Term &x, const Term &y) {
  Term r;
  r.c = x.c * y.c;
  size_t i = 0, j = 0;
  while (i < x.f.size() || j < y.f.size()) {
    if (j >= y.f.size() || (i < x.f.size() && x.f[i].first < y.f[j].first)) r.f.push_back(x.f[i++]);
    else if (i >= x.f.size() || y.f[j].first < x.f[i].first) r.f.push_back(y.f[j++]);
    else {
      r.f.push_back({x.f[i].first, x.f[i].second + y.f[j].second});
      ++i;
      ++j;
    }
  }
  return r;
}

struct Lowering {
  const RawDag &raw;
  const std::set<int> &fbound;
  int dim;
  bool cplx = false;
  std::vector<LNode> nodes;
  std::map<int, int> memo;   // raw id -> lowered id (as a root)
  std::map<int, int> memo2;  // raw id -> lowered id (as an operand)
  std::map<std::tuple<int, int, int, uint64_t, int>, int> cons;

  Lowering(const RawDag &r, const std::set<int> &fb, int d) : raw(r), fbound(fb), dim(d) {
    for (int i = 0; i < dim; ++i) {
      LNode v{L_VAR};
      v.n = i;
      nodes.push_back(v);
    }
  }
  int make(LK k, int a, int b, double c, int n) {
    auto key = std::make_tuple((int)k, a, b, dbits(c), n);
    auto it = cons.find(key);
    if (it != cons.end()) return it->second;
    LNode x{k};
    x.a = a;
    x.b = b;
    x.c = c;
    x.n = n;
    nodes.push_back(x);
    cons.emplace(key, (int)nodes.size() - 1);
    return (int)nodes.size() - 1;
  }
  int from_poly(Poly p) {
    normalize(p);
    if (p.empty()) return make(L_CONST, -1, -1, 0.0, 0);
    if (p.size() == 1 && p[0].f.empty()) return make(L_CONST, -1, -1, p[0].c, 0);
    if (p.size() == 1 && p[0].c == 1.0 && p[0].f.size() == 1 && p[0].f[0].second == 1) return p[0].f[0].first;
    LNode x{L_POLY};
    x.terms = p;
    nodes.push_back(x);
    return (int)nodes.size() - 1;
  }
  // node id = exp(q*log a), i.e. a real power a^q (R_POWR below): base a and exponent q
  bool as_real_power(int id, int &base, double &q) const {
    if (id < dim || nodes[id].k != L_EXP) return false;
    const LNode &arg = nodes[nodes[id].a];
    if (arg.k != L_POLY || arg.terms.size() != 1 || arg.terms[0].f.size() != 1 || arg.terms[0].f[0].second != 1) return false;
    const int ll = arg.terms[0].f[0].first;
    if (ll < dim || nodes[ll].k != L_LOG) return false;
    base = nodes[ll].a;
    q = arg.terms[0].c;
    return true;
  }
  // a variable, or a product of variables with coefficient 1: positive on the integration domain (0,1)^n
  bool variable_monomial(int id, Term &m) const {
    if (id < dim) {
      m = Term{1.0, {{id, 1}}};
      return true;
    }
    const LNode &n = nodes[id];
    if (n.k != L_POLY || n.terms.size() != 1 || n.terms[0].c != 1.0) return false;
    for (auto &fe : n.terms[0].f)
      if (fe.first >= dim) return false;
    m = n.terms[0];
    return true;
  }
  // Real arithmetic only: x_i^q * x_j^q -> (x_i x_j)^q for variables (and products of variables), one
  // log and one exp instead of one pair per factor.  The variables are positive on the integration
  // domain, the open unit cube (R2: u in (0,1)), where the two forms are the same function;
  // a caller of fiesta_eval_points with x <= 0 gets NaN from either unless an even number of the
  // merged variables is negative.  Not done in complex mode (branch cuts).
  void merge_real_powers(Term &t) {
    if (cplx) return;
    for (;;) {
      int i0 = -1, i1 = -1;
      for (size_t i = 0; i < t.f.size() && i1 < 0; ++i) {
        int bi;
        double qi;
        Term mi;
        if (t.f[i].second != 1 || !as_real_power(t.f[i].first, bi, qi) || !variable_monomial(bi, mi)) continue;
        for (size_t j = i + 1; j < t.f.size(); ++j) {
          int bj;
          double qj;
          Term mj;
          if (t.f[j].second != 1 || !as_real_power(t.f[j].first, bj, qj) || qj != qi || !variable_monomial(bj, mj)) continue;
          i0 = (int)i;
          i1 = (int)j;
          break;
        }
      }
      if (i1 < 0) return;
      int b0, b1;
      double q, q1;
      Term m0, m1;
      as_real_power(t.f[i0].first, b0, q);
      as_real_power(t.f[i1].first, b1, q1);
      variable_monomial(b0, m0);
      variable_monomial(b1, m1);
      const int prod = from_poly(Poly{mul_terms(m0, m1)});
      const int ll = make(L_LOG, prod, -1, 0, 0);
      const int arg = from_poly(Poly{Term{q, {{ll, 1}}}});
      const int e = make(L_EXP, arg, -1, 0, 0);
      t.f.erase(t.f.begin() + i1);
      t.f.erase(t.f.begin() + i0);
      Term one{1.0, {{e, 1}}};
      const double c = t.c;
      t = mul_terms(t, one);
      t.c = c;
    }
  }
  Poly atom_poly(int lid) {
    if (nodes[lid].k == L_CONST) {
      if (nodes[lid].c == 0.0) return Poly{};
      return Poly{Term{nodes[lid].c, {}}};
    }
    return Poly{Term{1.0, {{lid, 1}}}};
  }
  int lower(int rid) {
    auto it = memo.find(rid);
    if (it != memo.end()) return it->second;
    int lid = from_poly(poly_of(rid, true));
    memo[rid] = lid;
    return lid;
  }
  Poly poly_of(int rid, bool top) {
    const RNode &r = raw.nodes[rid];
    if (r.k == R_CONST) return r.c == 0.0 ? Poly{} : Poly{Term{r.c, {}}};
    if (r.k == R_VAR) return Poly{Term{1.0, {{r.n, 1}}}};
    if (!top && fbound.count(rid)) return atom_poly(lower(rid));
    switch (r.k) {
      case R_NEG: {
        Poly p = poly_of(r.a, false);
        for (auto &t : p) t.c = -t.c;
        return p;
      }
      case R_ADD:
      case R_SUB: {
        Poly p = poly_of(r.a, false), q = poly_of(r.b, false);
        for (auto &t : q) {
          if (r.k == R_SUB) t.c = -t.c;
          p.push_back(t);
        }
        normalize(p);
        return p;
      }
      case R_MUL: {
        Poly p = poly_of(r.a, false), q = poly_of(r.b, false);
        if (p.empty() || q.empty()) return Poly{};
        if (p.size() > 1 && q.size() > 1) {  // never expand polynomial x polynomial
          Poly pa = atom_poly(from_poly(p)), qa = atom_poly(from_poly(q));
          return Poly{mul_terms(pa[0], qa[0])};
        }
        const Poly &mono = p.size() == 1 ? p : q;
        const Poly &other = p.size() == 1 ? q : p;
        Poly out;
        for (auto &t : other) {
          out.push_back(mul_terms(mono[0], t));
          merge_real_powers(out.back());
        }
        normalize(out);
        return out;
      }
      case R_DIV: {
        Poly q = poly_of(r.b, false);
        Poly p = poly_of(r.a, false);
        if (q.size() == 1 && q[0].f.empty()) {  // division by a constant: exact per coefficient
          for (auto &t : p) t.c = t.c / q[0].c;
          return p;
        }
        int la = from_poly(p), lb = from_poly(q);
        return atom_poly(make(L_DIV, la, lb, 0, 0));
      }
      case R_POWI: {
        Poly p = poly_of(r.a, false);
        int n = r.n;
        if (n == 0) return Poly{Term{1.0, {}}};
        if (n == 1) return p;
        if (p.empty()) {
          if (n > 0) return Poly{};
          return Poly{Term{INFINITY, {}}};
        }
        bool small = true;  // a monomial stays a monomial while its exponents are small; p[x[1],1000] goes
        if (p.size() == 1)   // through L_POWI (square and multiply) instead of 999 multiplications
          for (auto &fe : p[0].f) small = small && (long)fe.second * n <= 8;
        if (p.size() == 1 && n > 0 && small) {
          Term t = p[0];
          double c = t.c;
          for (int i = 1; i < n; ++i) c *= t.c;  // repeated multiplication (R9)
          t.c = c;
          for (auto &fe : t.f) fe.second *= n;
          return Poly{t};
        }
        int la = from_poly(p);
        if (nodes[la].k == L_CONST) {
          double c = nodes[la].c, v = c;
          for (int i = 1; i < std::abs(n); ++i) v *= c;
          if (n < 0) v = 1.0 / v;
          return v == 0.0 ? Poly{} : Poly{Term{v, {}}};
        }
        if (n > 0 && n <= 4) return Poly{Term{1.0, {{la, n}}}};
        return atom_poly(make(L_POWI, la, -1, 0, n));
      }
      case R_POWR: {
        int la = lower_inner(r.a);
        if (r.c == 0.5) return atom_poly(make(L_SQRT, la, -1, 0, 0));
        int ll = make(L_LOG, la, -1, 0, 0);
        int arg = from_poly(Poly{Term{r.c, {{ll, 1}}}});
        return atom_poly(make(L_EXP, arg, -1, 0, 0));
      }
      case R_LOG:
        return atom_poly(make(L_LOG, lower_inner(r.a), -1, 0, 0));
      default:
        break;
    }
    fail(FIESTA_E_PARSE, "internal: unknown raw node");
  }
  int lower_inner(int rid) {  // an operand that becomes an opaque value
    if (fbound.count(rid)) return lower(rid);
    auto it = memo2.find(rid);
    if (it != memo2.end()) return it->second;
    int lid = from_poly(poly_of(rid, false));
    memo2[rid] = lid;
    return lid;
  }
};

// ------------------------------------------------------------------------------ emitter
struct Emitter {
  std::vector<LNode> &nodes;
  int dim;
  std::vector<fx_ins> code;
  bool sfree[FX_NS];
  std::vector<int> mfree;
  int mbase, mhigh;
  int s_high = 0;

  Emitter(std::vector<LNode> &n, int d, int mem_base) : nodes(n), dim(d), mbase(mem_base), mhigh(mem_base) {
    for (auto &b : sfree) b = true;
  }
  void ins(int op, int aux = 0, double imm = 0.0) {
    fx_ins i;
    i.op = (uint16_t)op;
    i.aux = (uint16_t)aux;
    i.pad = 0;
    i.imm = imm;
    code.push_back(i);
  }
  Opnd alloc_temp() {
    Opnd o;
    for (int j = 0; j < FX_NS; ++j)
      if (sfree[j]) {
        sfree[j] = false;
        s_high = std::max(s_high, j + 1);
        o.kind = Opnd::REG;
        o.idx = FX_REG_S(j);
        return o;
      }
    o.kind = Opnd::MEM;
    if (!mfree.empty()) {
      o.idx = mfree.back();
      mfree.pop_back();
    } else {
      o.idx = mhigh++;
      if (mhigh > 4096) fail(FIESTA_E_TOOBIG, "expression needs more than 4096 spill slots");
    }
    return o;
  }
  void free_temp(const Opnd &o) {
    if (o.kind == Opnd::REG) sfree[o.idx - FX_NXMAX] = true;
    else if (o.kind == Opnd::MEM) mfree.push_back(o.idx);
  }
  int lvl = 0;  // accumulator level the arithmetic helpers act on (0 outside horner())
  int LR(int base, const Opnd &o) const { return base + lvl * FX_NR + o.idx; }
  Opnd alloc_mem_temp() {
    Opnd o;
    o.kind = Opnd::MEM;
    if (!mfree.empty()) {
      o.idx = mfree.back();
      mfree.pop_back();
    } else {
      o.idx = mhigh++;
      if (mhigh > 4096) fail(FIESTA_E_TOOBIG, "expression needs more than 4096 spill slots");
    }
    return o;
  }
  void store(const Opnd &o) {  // from level 0 (registers) or any level (memory)
    if (o.kind == Opnd::REG) {
      if (lvl != 0) fail(FIESTA_E_ARG, "internal: register store from a nested level");
      ins(FX_ST_S + (o.idx - FX_NXMAX));
    } else
      ins(FX_STM + lvl, o.idx);
  }
  // -- A[lvl] <op> operand helpers
  void load(const Opnd &o) {
    if (o.kind == Opnd::IMM) ins(FX_LDC + lvl, 0, o.c);
    else if (o.kind == Opnd::REG) ins(LR(FX_LD_R, o));
    else ins(FX_LDM + lvl, o.idx);
  }
  void mul(const Opnd &o) {
    if (o.kind == Opnd::IMM) {
      if (o.c != 1.0) ins(FX_MULC + lvl, 0, o.c);
    } else if (o.kind == Opnd::REG) ins(LR(FX_MUL_R, o));
    else ins(FX_MULM + lvl, o.idx);
  }
  void add(const Opnd &o) {
    if (o.kind == Opnd::IMM) {
      if (o.c != 0.0) ins(FX_ADDC + lvl, 0, o.c);
    } else if (o.kind == Opnd::REG) ins(LR(FX_ADD_R, o));
    else ins(FX_ADDM + lvl, o.idx);
  }
  void div(const Opnd &o) {  // A = A / o   (level 0)
    if (o.kind == Opnd::IMM) ins(FX_DIVC, 0, o.c);
    else if (o.kind == Opnd::REG) ins(FX_DIV_R + o.idx);
    else ins(FX_DIVM, o.idx);
  }
  void rdiv(const Opnd &o) {  // A = o / A   (level 0)
    if (o.kind == Opnd::IMM) ins(FX_RDIVC, 0, o.c);
    else if (o.kind == Opnd::REG) ins(FX_RDIV_R + o.idx);
    else ins(FX_RDIVM, o.idx);
  }
  void fma_a(const Opnd &m, const Opnd &addend) {  // A = A*m + addend ; m is REG or MEM
    if (m.kind == Opnd::REG) {
      if (addend.kind == Opnd::IMM) ins(LR(FX_FMA_AR_C, m), 0, addend.c);
      else if (addend.kind == Opnd::MEM) ins(LR(FX_FMA_AR_M, m), addend.idx);
      else {
        ins(LR(FX_MUL_R, m));
        add(addend);
      }
    } else {
      if (addend.kind == Opnd::IMM) ins(FX_FMA_AM_C + lvl, m.idx, addend.c);
      else {
        ins(FX_MULM + lvl, m.idx);
        add(addend);
      }
    }
  }
  void fma_into_a(const Opnd &m, double c) {  // A = m*c + A
    if (m.kind == Opnd::REG) ins(LR(FX_FMA_RC_A, m), 0, c);
    else ins(FX_FMA_MC_A + lvl, m.idx, c);
  }
  void mulc_load(const Opnd &m, double c) {  // A = c*m
    if (m.kind == Opnd::REG) {
      if (c == 1.0) ins(LR(FX_LD_R, m));
      else ins(LR(FX_MULC_R, m), 0, c);
    } else {
      ins(FX_LDM + lvl, m.idx);
      if (c != 1.0) ins(FX_MULC + lvl, 0, c);
    }
  }

  Opnd operand_of(int id) {
    Opnd o;
    if (id < dim) {
      o.kind = Opnd::REG;
      o.idx = id;
      return o;
    }
    if (nodes[id].k == L_CONST) {
      o.kind = Opnd::IMM;
      o.c = nodes[id].c;
      return o;
    }
    if (nodes[id].mat) return nodes[id].loc;
    return o;  // NONE
  }
  bool available(int id) { return operand_of(id).kind != Opnd::NONE; }

  void count_uses(int id) {
    LNode &n = nodes[id];
    n.uses++;
    if (n.uses > 1) return;
    for (int c : children(id)) count_uses(c);
  }
  std::vector<int> children(int id) {
    const LNode &n = nodes[id];
    std::vector<int> out;
    if (n.k == L_POLY) {
      std::set<int> seen;
      for (auto &t : n.terms)
        for (auto &fe : t.f)
          if (fe.first >= dim && seen.insert(fe.first).second) out.push_back(fe.first);
    } else if (n.k == L_DIV) {
      out.push_back(n.a);
      out.push_back(n.b);
    } else if (n.k == L_LOG || n.k == L_EXP || n.k == L_POWI || n.k == L_SQRT) {
      out.push_back(n.a);
    }
    return out;
  }
  void consume(int id) {
    if (id < dim) return;
    LNode &n = nodes[id];
    if (n.k == L_CONST) return;
    if (--n.rem == 0 && n.mat) {
      free_temp(n.loc);
      n.mat = false;
      n.loc = Opnd{};
    }
  }
  void materialize_from_a(int id) {
    LNode &n = nodes[id];
    n.loc = alloc_temp();
    n.mat = true;
    store(n.loc);
  }
  // value of node id -> A.  Multi-use nodes are stored on first evaluation.
  void value_to_a(int id) {
    Opnd o = operand_of(id);
    if (o.kind != Opnd::NONE) {
      load(o);
      return;
    }
    emit(id);
    if (nodes[id].rem > 1) materialize_from_a(id);
  }
  void ensure_available(int id) {
    if (available(id)) return;
    emit(id);
    materialize_from_a(id);
  }

  void emit(int id) {
    LNode &n = nodes[id];
    switch (n.k) {
      case L_VAR:
      case L_CONST:
        load(operand_of(id));
        return;
      case L_LOG:
      case L_EXP:
      case L_SQRT:
        value_to_a(n.a);
        consume(n.a);
        ins(n.k == L_LOG ? FX_LOG : n.k == L_EXP ? FX_EXP : FX_SQRT);
        return;
      case L_POWI: {
        value_to_a(n.a);
        int e = std::abs(n.n);
        // square-and-multiply from the top bit; the base is kept in a temp when needed
        int top = 0;
        for (int b = 0; b < 31; ++b)
          if (e >> b & 1) top = b;
        bool need_base = (e & (e - 1)) != 0;
        Opnd base = operand_of(n.a);
        bool own = false;
        if (need_base && base.kind == Opnd::NONE) {
          base = alloc_temp();
          store(base);
          own = true;
        }
        for (int b = top - 1; b >= 0; --b) {
          ins(FX_SQR);
          if (e >> b & 1) mul(base);
        }
        if (own) free_temp(base);
        consume(n.a);
        if (n.n < 0) ins(FX_RDIVC, 0, 1.0);
        return;
      }
      case L_DIV: {
        int a = n.a, b = n.b;
        if (available(b)) {
          value_to_a(a);
          div(operand_of(b));
        } else if (available(a)) {
          value_to_a(b);
          rdiv(operand_of(a));
        } else {
          ensure_available(b);
          value_to_a(a);
          div(operand_of(b));
        }
        consume(a);
        consume(b);
        return;
      }
      case L_POLY:
        emit_poly(id);
        return;
    }
  }

  void emit_poly(int id) {
    const Poly terms = nodes[id].terms;  // copy: nodes may be touched while emitting children
    std::vector<int> atoms = children(id);
    if (terms.size() == 1) {
      // pure product: one not-yet-computed single-use atom may be computed last and stay in A
      const Term &t = terms[0];
      int in_a = -1;
      for (auto &fe : t.f)
        if (fe.first >= dim && fe.second == 1 && !available(fe.first) && in_a < 0) in_a = fe.first;
      for (int a : atoms)
        if (a != in_a) ensure_available(a);
      bool started = false;
      if (in_a >= 0) {
        value_to_a(in_a);
        if (t.c != 1.0) ins(FX_MULC, 0, t.c);
        started = true;
      }
      for (auto &fe : t.f) {
        if (fe.first == in_a) continue;
        Opnd o = operand_of(fe.first);
        for (int e = 0; e < fe.second; ++e) {
          if (!started) {
            mulc_load(o, t.c);
            started = true;
          } else
            mul(o);
        }
      }
      for (int a : atoms) consume(a);
      return;
    }
    for (int a : atoms) ensure_available(a);
    horner(terms);
    for (int a : atoms) consume(a);
  }

  // p = v*q + r
  static void split(const Poly &terms, int v, Poly &q, Poly &r) {
    for (auto &t : terms) {
      bool has = false;
      Term u;
      u.c = t.c;
      for (auto &fe : t.f) {
        if (fe.first == v) {
          has = true;
          if (fe.second > 1) u.f.push_back({fe.first, fe.second - 1});
        } else
          u.f.push_back(fe);
      }
      (has ? q : r).push_back(u);
    }
  }
  static int most_frequent(const Poly &terms) {
    std::map<int, int> cnt;
    for (auto &t : terms)
      for (auto &fe : t.f) cnt[fe.first]++;
    int v = -1, best = 0;
    for (auto &kv : cnt)
      if (kv.second > best) {
        best = kv.second;
        v = kv.first;
      }
    return v;
  }
  // FP64-pipe cost of what horner() emits for `terms`, in issue slots of the native tier: a multiply
  // or an FMA with two register operands 1, an FMA that reads three registers (the fold A[d] =
  // A[d+1]*v + A[d]) 1.5 -- a three-operand DFMA issues at 2/3 rate on sm_100a.
  // `v` >= 0: factor out v at this node.  Below (and here if v < 0): the best of all atoms for `look`
  // more levels, then the greedy rule (the atom dividing most terms).
  static double cost(const Poly &terms, int v, int look) {
    if (terms.empty()) return 0.0;
    if (terms.size() == 1) {
      int nf = 0;
      for (auto &fe : terms[0].f) nf += fe.second;
      return (double)nf;
    }
    if (v < 0) {
      if (look <= 0 || terms.size() <= 2) v = most_frequent(terms);
      else return best_variable(terms, look).second;
    }
    Poly q, r;
    split(terms, v, q, r);
    const int lk = look - 1;
    if (r.empty()) return cost(q, -1, lk) + 1.0;
    const bool q_const = q.size() == 1 && q[0].f.empty();
    const bool r_const = r.size() == 1 && r[0].f.empty();
    if (q_const) return cost(r, -1, lk) + 1.0;
    if (r_const) return cost(q, -1, lk) + 1.0;
    if (r.size() == 1 && r[0].f.size() == 1 && r[0].f[0].second == 1) return cost(q, -1, lk) + 2.0;
    if (q.size() == 1) return cost(r, -1, lk) + cost(q, -1, 0) + 1.0;  // monomial q: muls, then the fold with an immediate
    return cost(r, -1, lk) + cost(q, -1, lk) + 1.5;
  }
  // the FX_HORNER_CAND atoms that divide most terms are tried as the variable to factor out
  static std::pair<int, double> best_variable(const Poly &terms, int look) {
    std::map<int, int> cnt;
    for (auto &t : terms)
      for (auto &fe : t.f) cnt[fe.first]++;
    std::vector<std::pair<int, int>> cand;  // (-count, atom): most frequent first, ties by atom id
    for (auto &kv : cnt) cand.push_back({-kv.second, kv.first});
    std::sort(cand.begin(), cand.end());
    if (terms.size() <= 3 || cand.size() == 1) return {cand[0].second, 0.0};
    int best_v = -1;
    double best_c = 0.0;
    for (size_t i = 0; i < cand.size() && i < FX_HORNER_CAND; ++i) {
      if (-cand[i].first < 2 && i > 0) break;
      const double c = cost(terms, cand[i].second, look);
      if (best_v < 0 || c < best_c - 1e-9) {
        best_v = cand[i].second;
        best_c = c;
      }
    }
    return {best_v, best_c};
  }
  // FX_HORNER_LOOK levels of look-ahead over the greedy rule at every node that is emitted
  static int choose_variable(const Poly &terms) { return best_variable(terms, FX_HORNER_LOOK).first; }

  // Multivariate Horner: p = v*q + r, v chosen by choose_variable.
  void horner(const Poly &terms) {
    if (terms.empty()) {
      ins(FX_LDC + lvl, 0, 0.0);
      return;
    }
    if (terms.size() == 1) {
      const Term &t = terms[0];
      if (t.f.empty()) {
        ins(FX_LDC + lvl, 0, t.c);
        return;
      }
      bool started = false;
      for (auto &fe : t.f) {
        Opnd o = operand_of(fe.first);
        for (int e = 0; e < fe.second; ++e) {
          if (!started) {
            mulc_load(o, t.c);
            started = true;
          } else
            mul(o);
        }
      }
      return;
    }
    const int v = choose_variable(terms);
    Poly q, r;
    split(terms, v, q, r);
    Opnd vo = operand_of(v);
    if (r.empty()) {
      horner(q);
      mul(vo);
      return;
    }
    bool q_const = q.size() == 1 && q[0].f.empty();
    bool r_const = r.size() == 1 && r[0].f.empty();
    if (q_const) {  // p = c*v + r
      horner(r);
      fma_into_a(vo, q[0].c);
      return;
    }
    if (r_const) {  // p = q*v + c
      horner(q);
      Opnd c;
      c.kind = Opnd::IMM;
      c.c = r[0].c;
      fma_a(vo, c);
      return;
    }
    if (r.size() == 1 && r[0].f.size() == 1 && r[0].f[0].second == 1) {  // p = q*v + c*w
      horner(q);
      mul(vo);
      fma_into_a(operand_of(r[0].f[0].first), r[0].c);
      return;
    }
    // general case p = q*v + r: r stays in A[lvl] while q is evaluated one level up, then one
    // FMA folds them -- no store/reload of the partial result
    horner(r);
    if (lvl + 1 < FX_L && q.size() == 1) {
      // q = c*m, one monomial: the product m*v WITHOUT its coefficient, which enters at the fold as
      // the immediate of A[d] = A[d+1]*c + A[d] -- two register operands where the fold through
      // FMA_UP reads three (a three-operand DFMA issues at 2/3 rate on sm_100a)
      ++lvl;
      bool started = false;
      for (auto &fe : q[0].f) {
        Opnd o = operand_of(fe.first);
        for (int e = 0; e < fe.second; ++e) {
          if (!started) {
            mulc_load(o, 1.0);
            started = true;
          } else
            mul(o);
        }
      }
      mul(vo);
      --lvl;
      ins(FX_FMA_UPC + lvl, 0, q[0].c);
      return;
    }
    if (lvl + 1 < FX_L) {
      ++lvl;
      horner(q);
      if (vo.kind == Opnd::REG) {
        --lvl;
        ins(LR(FX_FMA_UP, vo));
      } else {
        mul(vo);
        --lvl;
        ins(FX_ADD_UP + lvl);
      }
      return;
    }
    Opnd t = alloc_mem_temp();  // nesting deeper than the accumulator stack: spill r to shared memory
    store(t);
    horner(q);
    fma_a(vo, t);
    free_temp(t);
  }
};

namespace {
bool in_fam(int op, int base, int n) { return op >= base && op < base + n; }
}

// FP64 flops of a program, counted as fma 2, mul/add 1, division 15, log/exp 40 (nominal weights for
// the library routines).  Complex programs (cplx): every instruction by the real operations of its
// handler (gen_interp_ptx.py): complex*complex 6, complex fma 8, fma with a real immediate 7 or 4,
// complex +- 2, division 6 + 15 + ..., log = log + atan2 (80), exp = exp + sincos (80).
void fill_info(const std::vector<fx_ins> &code, fiesta_compile_info &info, bool cplx) {
  for (auto &i : code) {
    int op = i.op;
    if (op == FX_END) continue;
    info.n_ir_ops++;
    bool fma = in_fam(op, FX_FMA_AR_C, 3 * FX_LR) || in_fam(op, FX_FMA_AR_M, FX_LR) || in_fam(op, FX_FMA_MC_A, 3 * FX_L);
    bool div = in_fam(op, FX_DIV_R, 2 * FX_NR) || op == FX_DIVC || op == FX_RDIVC || op == FX_DIVM || op == FX_RDIVM;
    bool move = in_fam(op, FX_LD_R, FX_LR) || in_fam(op, FX_ST_S, FX_NS) || in_fam(op, FX_LDC, FX_L) ||
                in_fam(op, FX_LDM, 2 * FX_L) || op == FX_OUT || op == FX_NEG;
    if (move) continue;
    info.n_fp64_ops++;
    if (fma) {
      info.n_fma++;
      if (!cplx) info.flops += 2;
      else if (in_fam(op, FX_FMA_RC_A, FX_LR) || in_fam(op, FX_FMA_MC_A, FX_L) || in_fam(op, FX_FMA_UPC, FX_L)) info.flops += 4;  // r*imm + a: 2 fma
      else if (in_fam(op, FX_FMA_AR_C, FX_LR) || in_fam(op, FX_FMA_AM_C, FX_L)) info.flops += 7;  // a*b + imm: 3 fma + mul
      else info.flops += 8;                                                                       // a*b + c: 4 fma
    } else if (div) {
      info.n_div++;
      if (!cplx) info.flops += 15;
      else if (op == FX_DIVC) info.flops += 30;
      else if (op == FX_RDIVC) info.flops += 3 + 15 + 2;
      else info.flops += 3 + 15 + 6 + 2;
    } else if (op == FX_LOG) {
      info.n_log++;
      info.flops += cplx ? 80 : 40;
    } else if (op == FX_EXP) {
      info.n_exp++;
      info.flops += cplx ? 80 : 40;
    } else if (op == FX_SQRT) {
      info.flops += cplx ? 40 : 15;
    } else if (!cplx) {
      info.flops += 1;
    } else if (in_fam(op, FX_MUL_R, FX_LR) || in_fam(op, FX_MUL_UP, FX_L) || in_fam(op, FX_MULM, FX_L) || op == FX_SQR) {
      info.flops += 6;  // complex * complex: 2 mul + 2 fma
    } else if (in_fam(op, FX_ADDC, FX_L) || op == FX_RSUBC) {
      info.flops += 1;  // real immediate added to the real part
    } else {
      info.flops += 2;  // componentwise: complex +-, times a real immediate
    }
  }
}

// Full expansion of a raw tree into monomials over x only (for the deformation polynomial F).
typedef std::map<std::vector<int>, double> XPoly;  // exponent vector -> coefficient

XPoly xmul(const XPoly &a, const XPoly &b) {
  XPoly out;
  for (auto &x : a)
    for (auto &y : b) {
      std::vector<int> e(x.first.size());
      for (size_t i = 0; i < e.size(); ++i) e[i] = x.first[i] + y.first[i];
      out[e] += x.second * y.second;
    }
  if (out.size() > 20000) fail(FIESTA_E_NOTPOLY, "deformation polynomial F expands to more than 20000 monomials");
  return out;
}

XPoly expand_full(const RawDag &raw, int rid, int dim) {
  const RNode &r = raw.nodes[rid];
  std::vector<int> zero(dim, 0);
  switch (r.k) {
    case R_CONST:
      return XPoly{{zero, r.c}};
    case R_VAR: {
      std::vector<int> e = zero;
      e[r.n] = 1;
      return XPoly{{e, 1.0}};
    }
    case R_NEG: {
      XPoly p = expand_full(raw, r.a, dim);
      for (auto &kv : p) kv.second = -kv.second;
      return p;
    }
    case R_ADD:
    case R_SUB: {
      XPoly p = expand_full(raw, r.a, dim), q = expand_full(raw, r.b, dim);
      for (auto &kv : q) p[kv.first] += (r.k == R_SUB ? -kv.second : kv.second);
      return p;
    }
    case R_MUL:
      return xmul(expand_full(raw, r.a, dim), expand_full(raw, r.b, dim));
    case R_DIV: {
      XPoly q = expand_full(raw, r.b, dim);
      if (q.size() != 1 || q.begin()->first != zero) fail(FIESTA_E_NOTPOLY, "deformation polynomial F must not divide by x");
      XPoly p = expand_full(raw, r.a, dim);
      for (auto &kv : p) kv.second /= q.begin()->second;
      return p;
    }
    case R_POWI: {
      if (r.n < 0) fail(FIESTA_E_NOTPOLY, "deformation polynomial F must have non-negative integer powers");
      XPoly out{{zero, 1.0}};
      XPoly base = expand_full(raw, r.a, dim);
      for (int i = 0; i < r.n; ++i) out = xmul(out, base);
      return out;
    }
    default:
      fail(FIESTA_E_NOTPOLY, "deformation polynomial F must be a polynomial in x (no logarithms or real powers)");
  }
}

Poly xpoly_derivative(const XPoly &p, int k, int l /* -1: first derivative only */) {
  Poly out;
  for (auto &kv : p) {
    std::vector<int> e = kv.first;
    double c = kv.second;
    if (e[k] == 0) continue;
    c *= e[k];
    e[k]--;
    if (l >= 0) {
      if (e[l] == 0) continue;
      c *= e[l];
      e[l]--;
    }
    if (c == 0.0) continue;
    Term t;
    t.c = c;
    for (int i = 0; i < (int)e.size(); ++i)
      if (e[i] > 0) t.f.push_back({i, e[i]});
    out.push_back(t);
  }
  return out;
}

}  // namespace

CompiledSector compile_sector(const char *const *texts, int K, int dim, bool is_complex, int deform_f_index,
                              double lambda) {
  if (dim < 1 || dim > FIESTA_MAX_DIM) fail(FIESTA_E_DIM, "dim must be in 1.." + std::to_string(FIESTA_MAX_DIM));
  if (K < 1 || K > FIESTA_MAX_ORDERS) fail(FIESTA_E_ARG, "n_orders must be in 1.." + std::to_string(FIESTA_MAX_ORDERS));
  RawDag raw;
  std::set<int> fbound;
  std::vector<int> roots(K), funcs0;
  for (int k = 0; k < K; ++k) {
    if (!texts || !texts[k]) fail(FIESTA_E_ARG, "NULL expression text");
    std::vector<int> funcs;
    parse_block(raw, texts[k], dim, fbound, "order " + std::to_string(k), funcs, roots[k]);
    if (k == 0) funcs0 = funcs;
  }
  CompiledSector cs;
  cs.K = K;
  cs.dim = dim;
  cs.is_complex = is_complex || deform_f_index > 0;
  cs.deform_on = deform_f_index > 0;
  cs.lambda = lambda;
  if (deform_f_index > 0 && !(lambda >= 0.0)) fail(FIESTA_E_ARG, "lambda must be >= 0 (PAPER.md:474: Im F(z) < 0 needs a positive deformation)");

  Lowering low(raw, fbound, dim);
  low.cplx = cs.is_complex;
  std::vector<int> lroots(K);
  for (int k = 0; k < K; ++k) lroots[k] = low.lower(roots[k]);
  {
    Emitter em(low.nodes, dim, 0);
    for (int k = 0; k < K; ++k) em.count_uses(lroots[k]);
    for (auto &n : low.nodes) n.rem = n.uses;
    for (int k = 0; k < K; ++k) {
      em.value_to_a(lroots[k]);
      em.consume(lroots[k]);
      em.ins(FX_OUT, k);
    }
    em.ins(FX_END);
    cs.main = em.code;
    cs.n_mem_main = em.mhigh;
    cs.info.n_reg_temps = em.s_high;
    cs.info.n_mem_slots = em.mhigh;
  }
  fill_info(cs.main, cs.info, cs.is_complex);

  if (cs.deform_on) {
    if (deform_f_index > (int)funcs0.size())
      fail(FIESTA_E_ARG, "deform_f_index " + std::to_string(deform_f_index) + " exceeds the number of f-lines");
    XPoly F = expand_full(raw, funcs0[deform_f_index - 1], dim);
    std::vector<LNode> dn;
    for (int i = 0; i < dim; ++i) {
      LNode v{L_VAR};
      v.n = i;
      dn.push_back(v);
    }
    int nout = dim + dim * (dim + 1) / 2;
    Emitter em(dn, dim, nout);
    int slot = 0;
    auto emit_out = [&](Poly p) {
      normalize(p);
      em.horner(p);
      em.ins(FX_STM, slot++);
    };
    for (int k = 0; k < dim; ++k) emit_out(xpoly_derivative(F, k, -1));
    for (int k = 0; k < dim; ++k)
      for (int l = k; l < dim; ++l) emit_out(xpoly_derivative(F, k, l));
    em.ins(FX_END);
    cs.deform = em.code;
    cs.n_mem_deform = em.mhigh;
    cs.info.n_deform_ops = (int)cs.deform.size() - 1;
    {  // F itself as a one-output complex program: what -testF evaluates at the deformed points
      Lowering lowf(raw, fbound, dim);
      lowf.cplx = true;
      const int rootf = lowf.lower(funcs0[deform_f_index - 1]);
      Emitter ef(lowf.nodes, dim, 0);
      ef.count_uses(rootf);
      for (auto &n : lowf.nodes) n.rem = n.uses;
      ef.value_to_a(rootf);
      ef.consume(rootf);
      ef.ins(FX_OUT, 0);
      ef.ins(FX_END);
      cs.testf = ef.code;
      cs.n_mem_testf = ef.mhigh;
    }
    fiesta_compile_info di{};
    fill_info(cs.deform, di, false);
    cs.info.flops += di.flops;
  }
  return cs;
}

std::string disassemble(const std::vector<fx_ins> &prog) {
  static const char *lr[] = {"A%d=%3$g*R%2$d", "A%d*=R%d", "A%d=A%1$d*R%d+%g", "A%d+=R%d*%g", "A%d+=A[+1]*R%d",
                             "A%d+=R%d", "A%d=R%d", "A%d=A%1$d*R%d+M"};
  static const char *lv[] = {"A%d=imm", "A%d+=imm", "A%d*=imm", "A%d+=A[+1]", "A%d*=A[+1]", "A%d=M", "M=A%d",
                             "A%d+=M", "A%d*=M", "A%d+=M*imm", "A%d=A%1$d*M+imm", "A%d+=A[+1]*imm"};
  static const char *r0[] = {"A-=R%d", "A=R%d-A", "A/=R%d", "A=R%d/A"};
  static const char *single[] = {"A=imm-A", "A/=imm", "A=imm/A", "A-=M", "A=M-A", "A/=M", "A=M/A", "A=-A", "A=A*A",
                                 "A=log A", "A=exp A", "A=sqrt A", "OUT", "END"};
  std::string out;
  char buf[200], b2[120];
  for (size_t pc = 0; pc < prog.size(); ++pc) {
    const fx_ins &i = prog[pc];
    int op = i.op;
    if (op < FX_LDC) {
      int f = op / FX_LR, d = (op % FX_LR) / FX_NR, r = op % FX_NR;
      std::snprintf(b2, sizeof b2, lr[f], d, r, i.imm);
    } else if (op < FX_SUB_R) {
      int f = (op - FX_LDC) / FX_L, d = (op - FX_LDC) % FX_L;
      std::snprintf(b2, sizeof b2, lv[f], d);
    } else if (op < FX_ST_S) {
      std::snprintf(b2, sizeof b2, r0[(op - FX_SUB_R) / FX_NR], (op - FX_SUB_R) % FX_NR);
    } else if (op < FX_RSUBC) {
      std::snprintf(b2, sizeof b2, "S%d=A", op - FX_ST_S);
    } else {
      std::snprintf(b2, sizeof b2, "%s", single[op - FX_RSUBC]);
    }
    std::snprintf(buf, sizeof buf, "%4zu  %-22s aux=%d imm=%.17g\n", pc, b2, i.aux, i.imm);
    out += buf;
  }
  return out;
}

}  // namespace fx
