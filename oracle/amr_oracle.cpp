// oracle/amr_oracle.cpp
//
// TEST INFRASTRUCTURE ONLY.  Plain CPU oracle of the consumer of `face_flux`: the coarse-fine flux
// fix-up and the fine -> coarse restriction that follow the fluid update of two adjacent AMR levels.  Only tests/ may load
// it.  Shares no code with paper_1103_3373_b200/csrc.
//
// PAPER.md:44 (section 2, step 5): "Store the fluxes across the boundaries of all grid patches ... only necessary in AMR";
// PAPER.md:137 (section 4.3): the "coarse-grid correction" the CPU applies after the GPU solver.  The paper gives no
// formula; this is the standard conservative fix-up it refers to, stated for the data layout of SURVEY.md 8(b)
// [reading S25, DESIGN.md]:
//   * a refined coarse patch (8^3 coarse cells) is covered by exactly one fine patch group (16^3 fine cells), so the six
//     outer boundary planes of that fine group (face_flux planes p = 3 d + s with s = 0 or 2) coincide with the six faces
//     of the coarse patch, each coarse face being covered by 2 x 2 fine faces;
//   * restriction: a covered coarse cell becomes the mean of its eight fine cells (volume average, uniform Cartesian cells),
//     summed in the fixed order ((x pairs) + (x pairs)) over y, then over z, times 1/8;
//   * flux fix-up: the unrefined coarse cell next to such a face was updated with the coarse flux F_c of that face (stored by
//     the coarse level's hydro_solve in ITS face_flux: the face is at f = 0, 8 or 16 of the coarse group, which is why the
//     mid-plane is stored, S16); conservation requires the area average of the fine fluxes instead, so
//         U <- U + sigma (dt_c / dh_c) (F_c - Fbar_f),   Fbar_f = ((f00 + f10) + (f01 + f11)) / 4,
//     sigma = +1 if the face is the cell's upper face along d (the fine group lies above), -1 if it is its lower face.
//     Fluxes are raw time-centred flux densities (S17); with sub-cycled fine steps the caller passes their dt-weighted
//     time average (oracle_flux_accum).
// Pins (tests/test_oracle_amr.py): exact conservation of the two-level composite totals on a periodic box (which fails by
// O(dt) without the fix-up, with a wrong sign, a wrong plane or in-plane order, or a wrong 1/4), the uniform-state identity
// (bitwise), restriction of dyadic linear data (exact).
#include <cstddef>

namespace {
constexpr int PS = 16, HP = 8;

// in-plane position of the face (a, b) of direction d inside a [16][16] plane: d=x -> [k][j], d=y -> [k][i], d=z -> [j][i]
inline size_t plane_at(int a, int b) { return (size_t)b * PS + a; }

struct CfFace { int fine_group, dir, fine_side, coarse_group, ci, cj, ck; };
struct Restrict { int fine_group, coarse_group, pi, pj, pk; };

template <class R>
void fluxfix(R* coarse_out, const R* coarse_flux, const R* fine_flux, const CfFace* faces, int nfaces, R dt_c, R dh_c) {
  const R nu = dt_c / dh_c;
  const size_t cell_n = (size_t)PS * PS * PS, plane_n = (size_t)PS * PS;
  for (int n = 0; n < nfaces; ++n) {
    const CfFace& f = faces[n];
    const int d = f.dir;
    const int c0[3] = {f.ci, f.cj, f.ck};
    const int layer = c0[d];                                  // coarse layer adjacent to the face
    const int cf = f.fine_side == 0 ? layer + 1 : layer;      // coarse face index: upper face of the layer if the fine group lies above
    const int s_c = cf / HP;                                  // cf in {0, 8, 16}
    const R sigma = f.fine_side == 0 ? R(1) : R(-1);
    const int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;       // in-plane axes, lower axis fastest
    const R* Fc = coarse_flux + ((size_t)f.coarse_group * 9 + (3 * d + s_c)) * 5 * plane_n;
    const R* Ff = fine_flux + ((size_t)f.fine_group * 9 + (3 * d + 2 * f.fine_side)) * 5 * plane_n;
    R* U = coarse_out + (size_t)f.coarse_group * 5 * cell_n;
    for (int q = 0; q < 5; ++q)
      for (int b = 0; b < HP; ++b)
        for (int a = 0; a < HP; ++a) {
          int c[3];
          c[d] = layer;
          c[t1] = c0[t1] + a;
          c[t2] = c0[t2] + b;
          const R fc = Fc[q * plane_n + plane_at(c[t1], c[t2])];
          const R* ff = Ff + q * plane_n;
          const R fbar = ((ff[plane_at(2 * a, 2 * b)] + ff[plane_at(2 * a + 1, 2 * b)]) +
                          (ff[plane_at(2 * a, 2 * b + 1)] + ff[plane_at(2 * a + 1, 2 * b + 1)])) * R(0.25);
          R& u = U[q * cell_n + ((size_t)c[2] * PS + c[1]) * PS + c[0]];
          u = u + sigma * nu * (fc - fbar);
        }
  }
}

template <class R> void restrict_groups(const R* fine_out, R* coarse_out, const Restrict* map, int n) {
  const size_t cell_n = (size_t)PS * PS * PS;
  for (int m = 0; m < n; ++m) {
    const Restrict& r = map[m];
    const R* F = fine_out + (size_t)r.fine_group * 5 * cell_n;
    R* C = coarse_out + (size_t)r.coarse_group * 5 * cell_n;
    for (int q = 0; q < 5; ++q)
      for (int k = 0; k < HP; ++k)
        for (int j = 0; j < HP; ++j)
          for (int i = 0; i < HP; ++i) {
            auto f = [&](int di, int dj, int dk) { return F[q * cell_n + ((size_t)(2 * k + dk) * PS + (2 * j + dj)) * PS + (2 * i + di)]; };
            const R lo = (f(0, 0, 0) + f(1, 0, 0)) + (f(0, 1, 0) + f(1, 1, 0));
            const R hi = (f(0, 0, 1) + f(1, 0, 1)) + (f(0, 1, 1) + f(1, 1, 1));
            C[q * cell_n + ((size_t)(r.pk + k) * PS + (r.pj + j)) * PS + (r.pi + i)] = (lo + hi) * R(0.125);
          }
  }
}

template <class R> void flux_accum(R* acc, const R* ff, size_t n, R w) {
  for (size_t i = 0; i < n; ++i) acc[i] = acc[i] + w * ff[i];
}
}  // namespace

extern "C" {
void oracle_fluxfix_f64(double* coarse_out, const double* coarse_flux, const double* fine_flux, const int* faces, int nfaces, double dt_c, double dh_c) {
  fluxfix<double>(coarse_out, coarse_flux, fine_flux, reinterpret_cast<const CfFace*>(faces), nfaces, dt_c, dh_c);
}
void oracle_fluxfix_f32(float* coarse_out, const float* coarse_flux, const float* fine_flux, const int* faces, int nfaces, float dt_c, float dh_c) {
  fluxfix<float>(coarse_out, coarse_flux, fine_flux, reinterpret_cast<const CfFace*>(faces), nfaces, dt_c, dh_c);
}
void oracle_restrict_f64(const double* fine_out, double* coarse_out, const int* map, int n) {
  restrict_groups<double>(fine_out, coarse_out, reinterpret_cast<const Restrict*>(map), n);
}
void oracle_restrict_f32(const float* fine_out, float* coarse_out, const int* map, int n) {
  restrict_groups<float>(fine_out, coarse_out, reinterpret_cast<const Restrict*>(map), n);
}
void oracle_flux_accum_f64(double* acc, const double* ff, long long n, double w) { flux_accum<double>(acc, ff, (size_t)n, w); }
void oracle_flux_accum_f32(float* acc, const float* ff, long long n, float w) { flux_accum<float>(acc, ff, (size_t)n, w); }
}
