// oracle/oracle.cpp  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, double-precision CPU photon tracker written from the paper
// (arXiv 2203.14354, /root/reference/PAPER.md, cited as P:<line>) and from the
// step list S1..S13 of SURVEY.md section 8(c) / DESIGN.md "Oracle".  It shares
// no source, header, table or helper with the CUDA library; only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
// may load it.  One photon at a time, one step at a time, in the order and
// notation of S1..S13.  The only speed-ups are (i) std::thread over disjoint
// photon ranges (photons are independent) and (ii) an optional
// top-down binary BVH for the first-hit query, which tests/ prove identical to
// the brute-force definition on random rays (pin P1).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"):
//   first hit      : P1  brute force on tiny meshes, analytic icosphere bound, BVH == brute force
//   absorption     : P2  exp(-R/L_abs) (BASELINE.json configs[0]); P2b competition closed forms
//   Fresnel        : P3  paper's printed 6.5% / 4.6% / 11.2% / 88.8%; P4 TIR at 75 deg,
//                        critical angles, Brewster angle, Snell, R+T=1
//   Rayleigh       : P5  3/8(1+cos^2) (Fig. 13 "theoretical distribution"), <mu^2>=1/5, 2/3 acceptance
//   Lambert        : P6  pdf 2cos, <cos>=2/3 ; specular P7 incl. normal incidence
//   surfaces/fates : P8  integrating sphere f/(1-rho(1-f)); P9 conservation; P10 transmit sheet
//   Philox4x32-10  : published known-answer vectors (tests/golden/philox4x32_10_kat.txt)
//   emission (E1-E5): position laws (r^2, z, rho^3 uniform), isotropy, e.k = 0 and uniform azimuth of e, Gaussian spectrum with
//                        mean 174.8 nm / FWHM 10.2 nm (Table 2), two-exponential time profile with tau_1, tau_3, f_s
//                        (Table 2): closed-form CDFs by KS, moments (tests/test_oracle_emission.py)
//   thin film (F1-F6)  : surface "calculated using Fresnel equations from the specified complex index of refraction and surface
//                        thickness": d -> 0 equals the bare interface, lossless film R + T = 1, quarter- and half-wave
//                        layers, thick absorbing film -> |r12|^2 (silicon n = 0.81, k = 1.86 of Table 8 seen from LXe: 0.436),
//                        evanescent exit -> T = 0, against an independent characteristic-matrix computation
//                        (tests/test_oracle_film.py).  NOT yet part of orc_propagate: coefficients and the single event only.
//   parity unpinned: trajectories beyond what the closed forms above fix, and the paper's own
//                    absolute LCE / t90 numbers (need the DARWIN CAD model).
//
// Units: mm, ns, nm.  c = 299.792458 mm/ns.
#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <limits>
#include <thread>
#include <vector>

namespace {

constexpr double kC = 299.792458;  // mm/ns
constexpr double kInf = std::numeric_limits<double>::infinity();
constexpr double kTwoPi = 6.283185307179586476925286766559;

// fate codes (low 4 bits of flags) and history bits -- same numbering as include/darwinopt.h,
// restated here (no shared header).
enum : uint32_t {
  FATE_DETECTED = 0, FATE_BULK_ABSORBED = 1, FATE_SURFACE_ABSORBED = 2, FATE_ESCAPED = 3,
  FATE_TRUNCATED = 4, FATE_NAN_ABORT = 5,
  H_RAYLEIGH = 0x10, H_REFLECT_DIFFUSE = 0x20, H_REFLECT_SPECULAR = 0x40, H_SURFACE_TRANSMIT = 0x80,
  H_FRESNEL_REFLECT = 0x100, H_FRESNEL_REFRACT = 0x200, H_TIR = 0x400, H_FILM = 0x1000
};

struct V3 { double x, y, z; };
inline V3 operator+(V3 a, V3 b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
inline V3 operator-(V3 a, V3 b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
inline V3 operator*(double s, V3 a) { return {s * a.x, s * a.y, s * a.z}; }
inline double dot(V3 a, V3 b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
inline V3 cross(V3 a, V3 b) { return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x}; }
inline double norm(V3 a) { return std::sqrt(dot(a, a)); }
inline V3 unit(V3 a) { return (1.0 / norm(a)) * a; }
inline bool finite3(V3 a) { return std::isfinite(a.x) && std::isfinite(a.y) && std::isfinite(a.z); }

// ---------------------------------------------------------------- S12: Philox4x32-10 (Salmon et al., SC'11)
struct U4 { uint32_t v[4]; };
inline U4 philox4x32_10(U4 ctr, uint32_t k0, uint32_t k1) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  for (int r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)M0 * ctr.v[0];
    uint64_t p1 = (uint64_t)M1 * ctr.v[2];
    U4 n;
    n.v[0] = (uint32_t)(p1 >> 32) ^ ctr.v[1] ^ k0;
    n.v[1] = (uint32_t)p1;
    n.v[2] = (uint32_t)(p0 >> 32) ^ ctr.v[3] ^ k1;
    n.v[3] = (uint32_t)p0;
    ctr = n;
    k0 += W0;
    k1 += W1;
  }
  return ctr;
}
// u = ((x >> 9) + 0.5) * 2^-23, in (0,1); 24 significant bits, so exactly representable in fp32 and the
// fp32 kernel and this fp64 code see the same number (S12; reading R-rng: SURVEY's (x>>8) form
// needs 25 bits and is not fp32-exact).
inline double u01(uint32_t x) { return ((double)(x >> 9) + 0.5) * (1.0 / 8388608.0); }
struct Rand4 { double u[4]; };
inline Rand4 draw(uint64_t seed, uint64_t photon, uint32_t step, uint32_t block) {
  U4 c{{(uint32_t)photon, (uint32_t)(photon >> 32), step, block}};
  U4 r = philox4x32_10(c, (uint32_t)seed, (uint32_t)(seed >> 32));
  return {{u01(r.v[0]), u01(r.v[1]), u01(r.v[2]), u01(r.v[3])}};
}

// ---------------------------------------------------------------- scene
struct Table {  // [n_rows][n_lambda] on a uniform lambda grid, linear interpolation, clamped (S3, G13)
  int rows = 0, nl = 0;
  double l0 = 0, dl = 1;
  std::vector<double> a;
  double at(int row, double lambda) const {
    if (nl == 1) return a[(size_t)row * nl];
    double f = (lambda - l0) / dl;
    if (f <= 0) return a[(size_t)row * nl];
    if (f >= nl - 1) return a[(size_t)row * nl + nl - 1];
    int i = (int)std::floor(f);
    double w = f - i;
    double y0 = a[(size_t)row * nl + i], y1 = a[(size_t)row * nl + i + 1];
    if (std::isinf(y0) || std::isinf(y1)) return (w == 0) ? y0 : (std::isinf(y1) ? y1 : y0);
    return y0 + w * (y1 - y0);
  }
};

struct BvhNode { double lo[3], hi[3]; int left, right, first, count; };  // count>0: leaf

struct Scene {
  std::vector<V3> vert;
  std::vector<int32_t> idx, mat_in, mat_out, surf, chan;
  int64_t nt = 0;
  Table n_idx, l_abs, l_sca;           // materials
  Table p_det, p_rd, p_rs, p_tr;       // surfaces
  Table f_n, f_k, f_d;                 // thin-film surfaces: index, extinction, thickness (nm); same grid as the surfaces
  std::vector<int32_t> film_on;        // per surface: 1 = the surface is a film (F-model), empty = none
  std::vector<BvhNode> nodes;          // own binary BVH (optional)
  std::vector<int32_t> order;          // triangle ids in leaf order
};

// ---------------------------------------------------------------- S1: ray/triangle, double Moeller-Trumbore,
// both edges inclusive, d > 0.
inline bool hit_triangle(const Scene& s, int64_t t, V3 o, V3 d, double& dist) {
  V3 v0 = s.vert[s.idx[3 * t]], v1 = s.vert[s.idx[3 * t + 1]], v2 = s.vert[s.idx[3 * t + 2]];
  V3 e1 = v1 - v0, e2 = v2 - v0;
  V3 p = cross(d, e2);
  double det = dot(e1, p);
  if (det == 0.0) return false;
  double inv = 1.0 / det;
  V3 tv = o - v0;
  double u = dot(tv, p) * inv;
  if (u < 0.0 || u > 1.0) return false;
  V3 q = cross(tv, e1);
  double v = dot(d, q) * inv;
  if (v < 0.0 || u + v > 1.0) return false;
  double tt = dot(e2, q) * inv;
  if (!(tt > 0.0)) return false;
  dist = tt;
  return true;
}

struct Hit { int32_t tri = -1; double d = kInf; };
inline void consider(const Scene& s, int64_t t, V3 o, V3 d, int32_t exclude, Hit& best) {
  if (t == exclude) return;
  double dd;
  if (!hit_triangle(s, t, o, d, dd)) return;
  if (dd < best.d || (dd == best.d && t < best.tri)) { best.d = dd; best.tri = (int32_t)t; }  // tie -> lowest id
}

Hit first_hit_brute(const Scene& s, V3 o, V3 d, int32_t exclude) {
  Hit best;
  for (int64_t t = 0; t < s.nt; ++t) consider(s, t, o, d, exclude, best);
  return best;
}

// ---- own BVH: top-down, median split of centroids along the widest axis, leaves <= 4 triangles.
void tri_bounds(const Scene& s, int32_t t, double lo[3], double hi[3]) {
  for (int a = 0; a < 3; ++a) { lo[a] = kInf; hi[a] = -kInf; }
  for (int k = 0; k < 3; ++k) {
    V3 v = s.vert[s.idx[3 * (int64_t)t + k]];
    double c[3] = {v.x, v.y, v.z};
    for (int a = 0; a < 3; ++a) { lo[a] = std::min(lo[a], c[a]); hi[a] = std::max(hi[a], c[a]); }
  }
}
int build_node(Scene& s, std::vector<V3>& cen, int first, int count) {
  BvhNode n{};
  for (int a = 0; a < 3; ++a) { n.lo[a] = kInf; n.hi[a] = -kInf; }
  double clo[3] = {kInf, kInf, kInf}, chi[3] = {-kInf, -kInf, -kInf};
  for (int i = first; i < first + count; ++i) {
    double lo[3], hi[3];
    tri_bounds(s, s.order[i], lo, hi);
    V3 c = cen[s.order[i]];
    double cc[3] = {c.x, c.y, c.z};
    for (int a = 0; a < 3; ++a) {
      n.lo[a] = std::min(n.lo[a], lo[a]); n.hi[a] = std::max(n.hi[a], hi[a]);
      clo[a] = std::min(clo[a], cc[a]); chi[a] = std::max(chi[a], cc[a]);
    }
  }
  for (int a = 0; a < 3; ++a) {  // pad so that boundary hits are never lost to rounding of the slab test
    double pad = 1e-9 * (1.0 + std::max(std::fabs(n.lo[a]), std::fabs(n.hi[a])));
    n.lo[a] -= pad; n.hi[a] += pad;
  }
  n.first = first; n.count = 0; n.left = n.right = -1;
  int me = (int)s.nodes.size();
  s.nodes.push_back(n);
  int axis = 0;
  for (int a = 1; a < 3; ++a) if (chi[a] - clo[a] > chi[axis] - clo[axis]) axis = a;
  if (count <= 4 || !(chi[axis] > clo[axis])) { s.nodes[me].count = count; return me; }
  int mid = first + count / 2;
  auto key = [&](int32_t t) { V3 c = cen[t]; return axis == 0 ? c.x : (axis == 1 ? c.y : c.z); };
  std::nth_element(s.order.begin() + first, s.order.begin() + mid, s.order.begin() + first + count,
                   [&](int32_t a, int32_t b) { double ka = key(a), kb = key(b); return ka < kb || (ka == kb && a < b); });
  int l = build_node(s, cen, first, mid - first);
  int r = build_node(s, cen, mid, first + count - mid);
  s.nodes[me].left = l; s.nodes[me].right = r;
  return me;
}
inline bool slab(const BvhNode& n, const double o[3], const double d[3], double tmax) {
  double t0 = 0.0, t1 = tmax;
  for (int a = 0; a < 3; ++a) {
    if (d[a] == 0.0) { if (o[a] < n.lo[a] || o[a] > n.hi[a]) return false; continue; }
    double inv = 1.0 / d[a];
    double ta = (n.lo[a] - o[a]) * inv, tb = (n.hi[a] - o[a]) * inv;
    if (ta > tb) std::swap(ta, tb);
    t0 = std::max(t0, ta); t1 = std::min(t1, tb);
  }
  return t0 <= t1 * (1.0 + 1e-12) + 1e-12;
}
Hit first_hit_bvh(const Scene& s, V3 o, V3 d, int32_t exclude) {
  Hit best;
  if (s.nodes.empty()) return best;
  const double oo[3] = {o.x, o.y, o.z}, dd[3] = {d.x, d.y, d.z};
  int stack[128]; int sp = 0; stack[sp++] = 0;
  while (sp) {
    const BvhNode& n = s.nodes[stack[--sp]];
    if (!slab(n, oo, dd, best.d)) continue;   // best.d inclusive: equal-distance ties are still visited
    if (n.count > 0) { for (int i = n.first; i < n.first + n.count; ++i) consider(s, s.order[i], o, d, exclude, best); }
    else { stack[sp++] = n.left; stack[sp++] = n.right; }
  }
  return best;
}
inline Hit first_hit(const Scene& s, V3 o, V3 d, int32_t exclude, bool use_bvh) {
  return use_bvh ? first_hit_bvh(s, o, d, exclude) : first_hit_brute(s, o, d, exclude);
}

// ---------------------------------------------------------------- physics pieces
// Orthonormal tangent frame (a, b, w) about a unit vector w: a = normalize(ref x w), b = w x a, with
// ref = x-axis if |w.x| < 0.5 else y-axis.  (Any frame is equal in distribution; this one is written
// down so that the step-locked test S12 can be stated.)
inline void frame(V3 w, V3& a, V3& b) {
  V3 ref = (std::fabs(w.x) < 0.5) ? V3{1, 0, 0} : V3{0, 1, 0};
  a = unit(cross(ref, w));
  b = cross(w, a);
}

// S6 Rayleigh scattering (the Geant4 algorithm that "reproduces the theoretical distribution").
// Iteration j uses Philox block 1+j: u0 -> cos(theta) of k', u1 -> azimuth of k', u2 -> accept.
inline int rayleigh(V3& k, V3& e, uint64_t seed, uint64_t pid, uint32_t step) {
  for (int j = 0; j < 100000; ++j) {
    Rand4 r = draw(seed, pid, step, 1u + (uint32_t)j);
    double ct = 1.0 - 2.0 * r.u[0];
    double st = std::sqrt(std::max(0.0, 1.0 - ct * ct));
    double ph = kTwoPi * r.u[1];
    V3 kn{st * std::cos(ph), st * std::sin(ph), ct};      // isotropic new direction
    V3 eraw = e - dot(e, kn) * kn;                          // old polarisation projected perpendicular to k'
    double w = dot(eraw, eraw);                             // = 1 - (e.k')^2 = cos^2(angle between e and e')
    if (r.u[2] < w) { k = kn; e = (1.0 / std::sqrt(w)) * eraw; return j + 1; }
  }
  return -1;
}

// S7 diffuse (Lambert): block 1: u0 -> cos(theta)=sqrt(u0), u1 -> azimuth, u2 -> polarisation angle
inline void lambert(V3 nhat, V3& k, V3& e, const Rand4& r) {
  double ct = std::sqrt(r.u[0]);
  double st = std::sqrt(std::max(0.0, 1.0 - r.u[0]));
  double ph = kTwoPi * r.u[1];
  V3 a, b;
  frame(nhat, a, b);
  k = unit(ct * nhat + (st * std::cos(ph)) * a + (st * std::sin(ph)) * b);
  double psi = kTwoPi * r.u[2];
  frame(k, a, b);
  e = std::cos(psi) * a + std::sin(psi) * b;               // uniformly random transverse (G8)
}

// S7 specular: no plane of incidence needed, normal incidence is not special
inline void specular(V3 nhat, V3& k, V3& e) {
  k = unit(k - (2.0 * dot(k, nhat)) * nhat);
  e = unit(e - (2.0 * dot(e, nhat)) * nhat);
}

// S8 Fresnel between n1 (photon side) and n2; nhat faces the photon (k.nhat <= 0).
// Returns 0 = reflected, 1 = refracted, 2 = total internal reflection; R_out = reflection probability.
inline int fresnel(double n1, double n2, V3 nhat, V3& k, V3& e, double u, double& R_out) {
  double ci = -dot(k, nhat);
  V3 sv = cross(k, nhat);
  double si = norm(sv);
  V3 s; double Es, Ep;
  if (si < 1e-9) { s = e; Es = 1.0; Ep = 0.0; }            // normal incidence: whole amplitude tangential
  else { s = (1.0 / si) * sv; V3 p = cross(s, k); Es = dot(e, s); Ep = dot(e, p); }
  double st = (n1 / n2) * si;
  if (st >= 1.0) {                                          // total internal reflection
    R_out = 1.0;
    V3 kr = unit(k + (2.0 * ci) * nhat);
    e = unit(Es * s + Ep * cross(s, kr));                   // magnitudes kept, phases ignored (G9)
    k = kr;
    return 2;
  }
  double ct = std::sqrt(1.0 - st * st);
  double rs = (n1 * ci - n2 * ct) / (n1 * ci + n2 * ct);
  double rp = (n2 * ci - n1 * ct) / (n2 * ci + n1 * ct);
  double ts = 2.0 * n1 * ci / (n1 * ci + n2 * ct);
  double tp = 2.0 * n1 * ci / (n2 * ci + n1 * ct);
  double R = Es * Es * rs * rs + Ep * Ep * rp * rp;
  R_out = R;
  if (u < R) {
    V3 kr = unit(k + (2.0 * ci) * nhat);
    e = unit((rs * Es) * s + (rp * Ep) * cross(s, kr));
    k = kr;
    return 0;
  }
  double eta = n1 / n2;
  V3 kt = unit(eta * k + (eta * ci - ct) * nhat);
  e = unit((ts * Es) * s + (tp * Ep) * cross(s, kt));
  k = kt;
  return 1;
}

// ---------------------------------------------------------------- thin-film surface
// "Surface reflectivity in Chroma can either be explicitly specified ..., or calculated using Fresnel equations from the
// specified complex index of refraction and surface thickness."  Textbook single-film (Airy) summation: a film of complex index
// n2 = nf + i kf and thickness d between the photon's medium n1 (real) and the material behind the triangle n3 (real).
// [readings F-*]: amplitudes per polarisation r = (r12 + r23 E^2) / (1 + r12 r23 E^2), t = t12 t23 E / (1 + r12 r23 E^2),
// E = exp(i 2 pi d n2 cos(theta2) / lambda), cos(theta2) = sqrt(1 - (n1 sin(theta1) / n2)^2) with the root that decays into
// the film; T = |t|^2 n3 cos(theta3) / (n1 cos(theta1)), zero when the wave in medium 3 is evanescent; A = 1 - R - T is
// absorbed in the film.  Mixed polarisation by intensities, as in S8.
typedef std::complex<double> Cx;
struct FilmCoef { double Rs, Rp, Ts, Tp, abs_rs, abs_rp, abs_ts, abs_tp; };
inline FilmCoef film_coefficients(double n1, double nf, double kf, double d_nm, double n3, double lambda_nm, double c1) {
  const Cx n2(nf, kf);
  const double s1 = std::sqrt(std::max(0.0, 1.0 - c1 * c1));
  Cx c2 = std::sqrt(Cx(1.0, 0.0) - (n1 * s1 / n2) * (n1 * s1 / n2));
  if ((n2 * c2).imag() < 0.0 || ((n2 * c2).imag() == 0.0 && (n2 * c2).real() < 0.0)) c2 = -c2;   // decays / propagates into the film
  const double s3 = n1 * s1 / n3;
  const bool evanescent = s3 >= 1.0;
  const Cx c3 = evanescent ? Cx(0.0, std::sqrt(s3 * s3 - 1.0)) : Cx(std::sqrt(1.0 - s3 * s3), 0.0);
  const Cx E = std::exp(Cx(0.0, 1.0) * (2.0 * M_PI * d_nm / lambda_nm) * n2 * c2), E2 = E * E;
  // s: electric field normal to the plane of incidence
  const Cx rs12 = (n1 * c1 - n2 * c2) / (n1 * c1 + n2 * c2), rs23 = (n2 * c2 - n3 * c3) / (n2 * c2 + n3 * c3);
  const Cx ts12 = 2.0 * n1 * c1 / (n1 * c1 + n2 * c2), ts23 = 2.0 * n2 * c2 / (n2 * c2 + n3 * c3);
  // p: electric field in the plane of incidence
  const Cx rp12 = (n2 * c1 - n1 * c2) / (n2 * c1 + n1 * c2), rp23 = (n3 * c2 - n2 * c3) / (n3 * c2 + n2 * c3);
  const Cx tp12 = 2.0 * n1 * c1 / (n2 * c1 + n1 * c2), tp23 = 2.0 * n2 * c2 / (n3 * c2 + n2 * c3);
  const Cx rs = (rs12 + rs23 * E2) / (1.0 + rs12 * rs23 * E2), rp = (rp12 + rp23 * E2) / (1.0 + rp12 * rp23 * E2);
  const Cx ts = ts12 * ts23 * E / (1.0 + rs12 * rs23 * E2), tp = tp12 * tp23 * E / (1.0 + rp12 * rp23 * E2);
  const double flux = evanescent ? 0.0 : n3 * c3.real() / (n1 * c1);
  return {std::norm(rs), std::norm(rp), std::norm(ts) * flux, std::norm(tp) * flux, std::abs(rs), std::abs(rp), std::abs(ts), std::abs(tp)};
}
// The surface event: 0 reflected (specular), 1 transmitted into medium 3, 2 absorbed in the film.  nhat faces the photon.
inline int film(double n1, double nf, double kf, double d_nm, double n3, double lambda_nm, V3 nhat, V3& k, V3& e, double u,
                double& R_out, double& T_out) {
  double ci = -dot(k, nhat);
  V3 sv = cross(k, nhat);
  double si = norm(sv);
  V3 s; double Es, Ep;
  if (si < 1e-9) { s = e; Es = 1.0; Ep = 0.0; }            // normal incidence: whole amplitude tangential
  else { s = (1.0 / si) * sv; V3 p = cross(s, k); Es = dot(e, s); Ep = dot(e, p); }
  const FilmCoef f = film_coefficients(n1, nf, kf, d_nm, n3, lambda_nm, ci);
  const double R = Es * Es * f.Rs + Ep * Ep * f.Rp, T = Es * Es * f.Ts + Ep * Ep * f.Tp;
  R_out = R; T_out = T;
  if (u < R) {
    V3 kr = unit(k + (2.0 * ci) * nhat);
    e = unit((f.abs_rs * Es) * s + (f.abs_rp * Ep) * cross(s, kr));   // magnitudes kept, phases ignored (G9)
    k = kr;
    return 0;
  }
  if (u < R + T) {
    double eta = n1 / n3, ct = std::sqrt(std::max(0.0, 1.0 - eta * eta * si * si));
    V3 kt = unit(eta * k + (eta * ci - ct) * nhat);
    e = unit((f.abs_ts * Es) * s + (f.abs_tp * Ep) * cross(s, kt));
    k = kt;
    return 1;
  }
  return 2;
}


struct PhotonOut { uint32_t flags, steps; int32_t channel, last_tri; double t; V3 x, k, e; };

// ---------------------------------------------------------------- the loop S1..S11 for one photon
PhotonOut propagate_one(const Scene& s, V3 x, V3 k, V3 e, double lambda, double t, uint64_t seed, uint64_t pid,
                        int32_t max_steps, bool use_bvh) {
  PhotonOut o{};
  uint32_t hist = 0, step = 0;
  int32_t last_tri = -1, channel = -1;
  uint32_t fate = FATE_TRUNCATED;                            // S10: loop exit by count
  while ((int32_t)step < max_steps) {
    if (!(finite3(x) && finite3(k) && finite3(e) && std::isfinite(t))) { fate = FATE_NAN_ABORT; break; }  // S11
    Rand4 r0 = draw(seed, pid, step, 0);                     // [u_a, u_s, u_surface, u_fresnel]
    Hit h = first_hit(s, x, k, last_tri, use_bvh);           // S1
    if (h.tri < 0) { fate = FATE_ESCAPED; ++step; break; }   // G3
    int64_t T = h.tri;
    V3 v0 = s.vert[s.idx[3 * T]], v1 = s.vert[s.idx[3 * T + 1]], v2 = s.vert[s.idx[3 * T + 2]];
    V3 ng = unit(cross(v1 - v0, v2 - v0));
    int m1, m2; V3 nhat;                                     // S2
    if (dot(k, ng) > 0) { m1 = s.mat_in[T]; m2 = s.mat_out[T]; nhat = (-1.0) * ng; }
    else { m1 = s.mat_out[T]; m2 = s.mat_in[T]; nhat = ng; }
    double n1 = s.n_idx.at(m1, lambda), La = s.l_abs.at(m1, lambda), Ls = s.l_sca.at(m1, lambda);  // S3
    double da = std::isinf(La) ? kInf : -La * std::log(r0.u[0]);  // S4
    double ds = std::isinf(Ls) ? kInf : -Ls * std::log(r0.u[1]);
    if (da < ds && da < h.d) {
      x = x + da * k; t += da * n1 / kC; fate = FATE_BULK_ABSORBED; ++step; break;
    }
    if (ds < h.d) {
      x = x + ds * k; t += ds * n1 / kC;
      if (rayleigh(k, e, seed, pid, step) < 0) { fate = FATE_NAN_ABORT; ++step; break; }
      hist |= H_RAYLEIGH; last_tri = -1; ++step; continue;
    }
    x = x + h.d * k; t += h.d * n1 / kC; last_tri = h.tri;   // S4 third branch, S5
    int sf = s.surf[T];
    if (sf >= 0 && !s.film_on.empty() && s.film_on[sf]) {    // thin-film surface (second mode)
      double n3 = s.n_idx.at(m2, lambda), R, Tt;
      int oc = film(n1, s.f_n.at(sf, lambda), s.f_k.at(sf, lambda), s.f_d.at(sf, lambda), n3, lambda, nhat, k, e, r0.u[3], R, Tt);
      hist |= H_FILM;
      if (oc == 0) hist |= H_REFLECT_SPECULAR;
      else if (oc == 1) hist |= H_SURFACE_TRANSMIT;
      else {                                                 // absorbed in the film: detected with the surface's detect probability
        if (r0.u[2] < s.p_det.at(sf, lambda)) { fate = FATE_DETECTED; channel = s.chan[T]; }
        else fate = FATE_SURFACE_ABSORBED;
        ++step; break;
      }
    } else if (sf >= 0) {                                    // S7 explicit surface
      double pd = s.p_det.at(sf, lambda), prd = s.p_rd.at(sf, lambda), prs = s.p_rs.at(sf, lambda),
             ptr = s.p_tr.at(sf, lambda);
      double u = r0.u[2];
      if (u < pd) { fate = FATE_DETECTED; channel = s.chan[T]; ++step; break; }
      else if (u < pd + prd) { lambert(nhat, k, e, draw(seed, pid, step, 1)); hist |= H_REFLECT_DIFFUSE; }
      else if (u < pd + prd + prs) { specular(nhat, k, e); hist |= H_REFLECT_SPECULAR; }
      else if (u < pd + prd + prs + ptr) { hist |= H_SURFACE_TRANSMIT; }
      else { fate = FATE_SURFACE_ABSORBED; ++step; break; }
    } else {                                                 // S8 Fresnel
      double n2 = s.n_idx.at(m2, lambda), R;
      int oc = fresnel(n1, n2, nhat, k, e, r0.u[3], R);
      hist |= (oc == 1) ? H_FRESNEL_REFRACT : (oc == 2 ? (H_FRESNEL_REFLECT | H_TIR) : H_FRESNEL_REFLECT);
    }
    ++step;                                                  // S9
  }
  if (fate == FATE_TRUNCATED && !(finite3(x) && finite3(k) && finite3(e) && std::isfinite(t))) fate = FATE_NAN_ABORT;
  o.flags = fate | hist; o.steps = step; o.channel = channel; o.last_tri = last_tri; o.t = t; o.x = x; o.k = k; o.e = e;
  return o;
}

template <class F>
void parallel_for(int64_t n, int nthreads, F f) {
  if (nthreads <= 1 || n < 2) { f(0, 0, n); return; }
  nthreads = (int)std::min<int64_t>(nthreads, n);
  std::vector<std::thread> th;
  for (int i = 0; i < nthreads; ++i) {
    int64_t a = n * i / nthreads, b = n * (i + 1) / nthreads;
    th.emplace_back([=] { f(i, a, b); });
  }
  for (auto& t : th) t.join();
}

int set_table(Table& tb, int rows, int nl, double l0, double dl, const float* a) {
  tb.rows = rows; tb.nl = nl; tb.l0 = l0; tb.dl = dl;
  tb.a.assign((size_t)rows * nl, 0.0);
  for (size_t i = 0; i < tb.a.size(); ++i) tb.a[i] = (double)a[i];
  return 0;
}

}  // namespace

// =================================================================== C interface for ctypes (tests / bench)
// ---------------------------------------------------------------- emission
// One scintillation photon per id, drawn from Philox blocks 0..2 of the reserved step 0xFFFFFFFF (propagation steps are
// < 2^31, so the streams never meet).  P:144: "The emission spectrum is modeled as a Gaussian with a mean of 174.8 nm and a
// full width at half maximum of 10.2 nm.  The scintillation time profile is modeled by a two-component exponential decay
// function"; Table 2: tau_1 = 3.5 ns, tau_3 = 24 ns, f_s = 0.66 (NR) / 0.22 (ER).  P:191: photons "generated
// isotropically and uniformly" in the active region.  [readings, DESIGN.md E-*]: random transverse polarisation = normalize(k x r)
// for an independent isotropic r; the spectrum is not truncated (tables clamp); the singlet branch is taken when
// u < (float)f_s, the comparison the fp32 kernel makes.
struct Source {
  int shape;            // 0 point, 1 cylinder (axis z), 2 ball
  double c[3];          // point / centre of the cylinder axis at z0 / centre of the ball
  double radius;        // cylinder or ball radius
  double z0, z1;        // cylinder: z range
  double lambda_mean, lambda_sigma;   // nm; sigma = FWHM / (2 sqrt(2 ln 2))
  double t_start, tau1, tau3, f_singlet;
};
constexpr uint32_t kEmitStep = 0xFFFFFFFFu;
inline V3 isotropic(double u_cos, double u_phi) {
  double ct = 1.0 - 2.0 * u_cos, st = std::sqrt(std::max(0.0, 1.0 - ct * ct)), ph = 2.0 * M_PI * u_phi;
  return {st * std::cos(ph), st * std::sin(ph), ct};
}
inline void emit(const Source& s, uint64_t seed, uint64_t pid, V3& x, V3& k, V3& e, double& lambda, double& t) {
  const Rand4 a = draw(seed, pid, kEmitStep, 0), b = draw(seed, pid, kEmitStep, 1), c = draw(seed, pid, kEmitStep, 2);
  // E1 position
  if (s.shape == 1) {
    double r = s.radius * std::sqrt(a.u[0]), ph = 2.0 * M_PI * a.u[1];
    x = {s.c[0] + r * std::cos(ph), s.c[1] + r * std::sin(ph), s.z0 + (s.z1 - s.z0) * a.u[2]};
  } else if (s.shape == 2) {
    V3 d = isotropic(a.u[1], a.u[2]);
    double r = s.radius * std::cbrt(a.u[0]);
    x = {s.c[0] + r * d.x, s.c[1] + r * d.y, s.c[2] + r * d.z};
  } else {
    x = {s.c[0], s.c[1], s.c[2]};
  }
  // E2 direction, E3 polarisation
  k = isotropic(b.u[0], b.u[1]);
  V3 r = isotropic(b.u[2], b.u[3]);
  V3 kr = cross(k, r);
  if (dot(kr, kr) < 1e-12) { V3 a2, b2; frame(k, a2, b2); e = a2; }
  else e = unit(kr);
  // E4 wavelength (Box-Muller), E5 time
  lambda = s.lambda_mean + s.lambda_sigma * std::sqrt(-2.0 * std::log(c.u[0])) * std::cos(2.0 * M_PI * c.u[1]);
  const double tau = (c.u[2] < (double)(float)s.f_singlet) ? s.tau1 : s.tau3;
  t = s.t_start - tau * std::log(c.u[3]);
}

extern "C" {

// out: 11 arrays of n doubles in the order of dw_photons (px py pz kx ky kz ex ey ez wavelength t0)
void orc_emit(int shape, const double* c3, double radius, double z0, double z1, double lambda_mean, double lambda_sigma,
              double t_start, double tau1, double tau3, double f_singlet, uint64_t seed, uint64_t id_base, int64_t n, double* out) {
  Source s{shape, {c3[0], c3[1], c3[2]}, radius, z0, z1, lambda_mean, lambda_sigma, t_start, tau1, tau3, f_singlet};
  for (int64_t i = 0; i < n; ++i) {
    V3 x, k, e;
    double lambda, t;
    emit(s, seed, id_base + (uint64_t)i, x, k, e, lambda, t);
    const double v[11] = {x.x, x.y, x.z, k.x, k.y, k.z, e.x, e.y, e.z, lambda, t};
    for (int f = 0; f < 11; ++f) out[(size_t)f * n + i] = v[f];
  }
}

// out: Rs Rp Ts Tp
void orc_film_coefficients(double n1, double nf, double kf, double d_nm, double n3, double lambda_nm, double cos1, double out[4]) {
  FilmCoef f = film_coefficients(n1, nf, kf, d_nm, n3, lambda_nm, cos1);
  out[0] = f.Rs; out[1] = f.Rp; out[2] = f.Ts; out[3] = f.Tp;
}
int orc_film(double n1, double nf, double kf, double d_nm, double n3, double lambda_nm, const double nhat[3], double k[3], double e[3],
             double u, double RT[2]) {
  V3 kk{k[0], k[1], k[2]}, ee{e[0], e[1], e[2]};
  int oc = film(n1, nf, kf, d_nm, n3, lambda_nm, {nhat[0], nhat[1], nhat[2]}, kk, ee, u, RT[0], RT[1]);
  k[0] = kk.x; k[1] = kk.y; k[2] = kk.z; e[0] = ee.x; e[1] = ee.y; e[2] = ee.z;
  return oc;
}

void* orc_create() { return new Scene(); }
void orc_destroy(void* h) { delete (Scene*)h; }
int orc_hardware_threads() { return (int)std::max(1u, std::thread::hardware_concurrency()); }

int orc_set_materials(void* h, int n_mat, int n_lambda, double lambda0, double dlambda, const float* refr,
                      const float* abs_len, const float* scat_len) {
  Scene& s = *(Scene*)h;
  set_table(s.n_idx, n_mat, n_lambda, lambda0, dlambda, refr);
  set_table(s.l_abs, n_mat, n_lambda, lambda0, dlambda, abs_len);
  set_table(s.l_sca, n_mat, n_lambda, lambda0, dlambda, scat_len);
  return 0;
}
int orc_set_surfaces(void* h, int n_surf, int n_lambda, double lambda0, double dlambda, const float* det,
                     const float* rd, const float* rs, const float* tr) {
  Scene& s = *(Scene*)h;
  set_table(s.p_det, n_surf, n_lambda, lambda0, dlambda, det);
  set_table(s.p_rd, n_surf, n_lambda, lambda0, dlambda, rd);
  set_table(s.p_rs, n_surf, n_lambda, lambda0, dlambda, rs);
  set_table(s.p_tr, n_surf, n_lambda, lambda0, dlambda, tr);
  return 0;
}
int orc_set_films(void* h, int n_surf, int n_lambda, double lambda0, double dlambda, const int32_t* film_on, const float* nf,
                  const float* kf, const float* d_nm) {
  Scene& s = *(Scene*)h;
  s.film_on.assign(film_on, film_on + n_surf);
  set_table(s.f_n, n_surf, n_lambda, lambda0, dlambda, nf);
  set_table(s.f_k, n_surf, n_lambda, lambda0, dlambda, kf);
  set_table(s.f_d, n_surf, n_lambda, lambda0, dlambda, d_nm);
  return 0;
}
int orc_set_geometry(void* h, int64_t nv, const float* xyz, int64_t nt, const int32_t* idx, const int32_t* mat_in,
                     const int32_t* mat_out, const int32_t* surf, const int32_t* chan) {
  Scene& s = *(Scene*)h;
  s.vert.resize(nv);
  for (int64_t i = 0; i < nv; ++i) s.vert[i] = {xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2]};
  s.nt = nt;
  s.idx.assign(idx, idx + 3 * nt);
  s.mat_in.assign(mat_in, mat_in + nt); s.mat_out.assign(mat_out, mat_out + nt);
  s.surf.assign(surf, surf + nt); s.chan.assign(chan, chan + nt);
  s.nodes.clear(); s.order.clear();
  return 0;
}
int orc_build_bvh(void* h) {
  Scene& s = *(Scene*)h;
  s.nodes.clear();
  s.order.resize(s.nt);
  std::vector<V3> cen(s.nt);
  for (int64_t t = 0; t < s.nt; ++t) {
    s.order[t] = (int32_t)t;
    cen[t] = (1.0 / 3.0) * (s.vert[s.idx[3 * t]] + s.vert[s.idx[3 * t + 1]] + s.vert[s.idx[3 * t + 2]]);
  }
  if (s.nt > 0) build_node(s, cen, 0, (int)s.nt);
  return (int)s.nodes.size();
}

// rays as SoA float32 (the same arrays the GPU gets); exclude may be NULL. use_bvh: 0 brute force, 1 own BVH.
void orc_first_hit(void* h, int64_t n, const float* ox, const float* oy, const float* oz, const float* dx,
                   const float* dy, const float* dz, const int32_t* exclude, int use_bvh, int32_t* tri, double* dist,
                   int nthreads) {
  const Scene& s = *(Scene*)h;
  parallel_for(n, nthreads, [&](int, int64_t a, int64_t b) {
    for (int64_t i = a; i < b; ++i) {
      Hit hh = first_hit(s, {ox[i], oy[i], oz[i]}, {dx[i], dy[i], dz[i]}, exclude ? exclude[i] : -1, use_bvh != 0);
      tri[i] = hh.tri; dist[i] = hh.d;
    }
  });
}

// Photon batch in, per-photon results + histograms out (S13).  Any output pointer may be NULL.
// Histograms are ACCUMULATED into.  out_xyz / out_dir / out_pol are [3][n] double.
void orc_propagate(void* h, int64_t n, const float* px, const float* py, const float* pz, const float* kx,
                   const float* ky, const float* kz, const float* ex, const float* ey, const float* ez,
                   const float* wavelength, const float* t0, uint64_t id_base, uint64_t seed, int32_t max_steps,
                   int use_bvh, uint32_t* flags, int32_t* channel, double* t_out, uint32_t* steps, int32_t* last_tri,
                   double* out_xyz, double* out_dir, double* out_pol, int64_t n_chan, uint64_t* chan_count,
                   int64_t n_bins, double t_min, double dt, uint64_t* time_hist, uint64_t* fate_count,
                   uint64_t* total_steps, int nthreads) {
  const Scene& s = *(Scene*)h;
  nthreads = std::max(1, nthreads);
  std::vector<std::vector<uint64_t>> cc(nthreads), th(nthreads), fc(nthreads);
  std::vector<uint64_t> ts(nthreads, 0);
  parallel_for(n, nthreads, [&](int w, int64_t a, int64_t b) {
    cc[w].assign((size_t)std::max<int64_t>(n_chan, 0), 0); th[w].assign((size_t)std::max<int64_t>(n_bins, 0), 0);
    fc[w].assign(8, 0);
    for (int64_t i = a; i < b; ++i) {
      PhotonOut o = propagate_one(s, {px[i], py[i], pz[i]}, {kx[i], ky[i], kz[i]}, {ex[i], ey[i], ez[i]},
                                  wavelength[i], t0[i], seed, id_base + (uint64_t)i, max_steps, use_bvh != 0);
      if (flags) flags[i] = o.flags;
      if (channel) channel[i] = o.channel;
      if (t_out) t_out[i] = o.t;
      if (steps) steps[i] = o.steps;
      if (last_tri) last_tri[i] = o.last_tri;
      if (out_xyz) { out_xyz[i] = o.x.x; out_xyz[n + i] = o.x.y; out_xyz[2 * n + i] = o.x.z; }
      if (out_dir) { out_dir[i] = o.k.x; out_dir[n + i] = o.k.y; out_dir[2 * n + i] = o.k.z; }
      if (out_pol) { out_pol[i] = o.e.x; out_pol[n + i] = o.e.y; out_pol[2 * n + i] = o.e.z; }
      uint32_t fate = o.flags & 0xF;                          // S13 reductions: plain counting
      fc[w][fate] += 1; ts[w] += o.steps;
      if (fate == FATE_DETECTED) {
        if (o.channel >= 0 && o.channel < n_chan) cc[w][o.channel] += 1;
        if (n_bins > 0) {
          double fb = std::floor((o.t - t_min) / dt);
          int64_t bin = fb < 0 ? 0 : (fb > (double)(n_bins - 1) ? n_bins - 1 : (int64_t)fb);
          th[w][bin] += 1;
        }
      }
    }
  });
  for (int w = 0; w < nthreads; ++w) {
    if (cc[w].empty() && th[w].empty() && fc[w].empty()) continue;
    if (chan_count) for (size_t c = 0; c < cc[w].size(); ++c) chan_count[c] += cc[w][c];
    if (time_hist) for (size_t c = 0; c < th[w].size(); ++c) time_hist[c] += th[w][c];
    if (fate_count) for (size_t c = 0; c < fc[w].size(); ++c) fate_count[c] += fc[w][c];
    if (total_steps) total_steps[0] += ts[w];
  }
}

// ---- single pieces, exported so that each can be pinned on its own
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  U4 c{{ctr[0], ctr[1], ctr[2], ctr[3]}};
  U4 r = philox4x32_10(c, key[0], key[1]);
  for (int i = 0; i < 4; ++i) out[i] = r.v[i];
}
void orc_uniforms(uint64_t seed, uint64_t photon, uint32_t step, uint32_t block, double out[4]) {
  Rand4 r = draw(seed, photon, step, block);
  for (int i = 0; i < 4; ++i) out[i] = r.u[i];
}
int orc_rayleigh(double k[3], double e[3], uint64_t seed, uint64_t pid, uint32_t step) {
  V3 kk{k[0], k[1], k[2]}, ee{e[0], e[1], e[2]};
  int it = rayleigh(kk, ee, seed, pid, step);
  k[0] = kk.x; k[1] = kk.y; k[2] = kk.z; e[0] = ee.x; e[1] = ee.y; e[2] = ee.z;
  return it;
}
void orc_lambert(const double nhat[3], double k[3], double e[3], uint64_t seed, uint64_t pid, uint32_t step) {
  V3 kk{k[0], k[1], k[2]}, ee{e[0], e[1], e[2]};
  lambert({nhat[0], nhat[1], nhat[2]}, kk, ee, draw(seed, pid, step, 1));
  k[0] = kk.x; k[1] = kk.y; k[2] = kk.z; e[0] = ee.x; e[1] = ee.y; e[2] = ee.z;
}
void orc_specular(const double nhat[3], double k[3], double e[3]) {
  V3 kk{k[0], k[1], k[2]}, ee{e[0], e[1], e[2]};
  specular({nhat[0], nhat[1], nhat[2]}, kk, ee);
  k[0] = kk.x; k[1] = kk.y; k[2] = kk.z; e[0] = ee.x; e[1] = ee.y; e[2] = ee.z;
}
int orc_fresnel(double n1, double n2, const double nhat[3], double k[3], double e[3], double u, double* R) {
  V3 kk{k[0], k[1], k[2]}, ee{e[0], e[1], e[2]};
  int oc = fresnel(n1, n2, {nhat[0], nhat[1], nhat[2]}, kk, ee, u, *R);
  k[0] = kk.x; k[1] = kk.y; k[2] = kk.z; e[0] = ee.x; e[1] = ee.y; e[2] = ee.z;
  return oc;
}

}  // extern "C"
