// oracle/rta_oracle_image.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain single-threaded CPU definition of the first downstream RT-RECO step
// (SURVEY.md §8(f) NEXT-4): image cleaning and image moments per event, so that
// "event-level reconstruction parameters (but not the raw data)" leave the
// device (§2.2). The paper names the chain only — "calibration, the
// gamma/hadron separation, and the energy and direction reconstruction"
// (§4.1), RT-RECO being "a reduced version" focused on speed
// (§4.2) — and defines none of it, so the operation below is the
// builder's (readings R31-R35): a two-threshold neighbour cleaning
// followed by the intensity-weighted first and second moments of the surviving
// pixels (the classic image-parameter approach of imaging Cherenkov telescopes,
// restated here from its textbook definition).
//
// Per event e, with q[p] = charge[e][p], t[p] = time[e][p], pixel centres
// (x[p], y[p]) and up to six neighbours nbr[p][0..5] (-1 = none):
//
//   core[p]  = q[p] >= thr_picture                                   (fp32 compare; NaN fails)
//   keep[p]  = core[p] and some neighbour n of p has core[n]          (isolated core pixels drop)
//   edge[p]  = q[p] >= thr_boundary and some neighbour n of p has keep[n]
//   mask[p]  = keep[p] or edge[p]
//   n_pix    = number of pixels in the mask
//   size     = sum q                     over the mask
//   cog_x    = sum q x / size,  cog_y = sum q y / size
//   sxx      = sum q (x - cog_x)^2 / size, syy likewise, sxy = sum q (x-cog_x)(y-cog_y) / size
//   z        = sqrt((sxx - syy)^2 + 4 sxy^2)
//   length   = sqrt((sxx + syy + z) / 2),  width = sqrt(max(0, (sxx + syy - z) / 2))
//   psi      = atan2(2 sxy, sxx - syy) / 2         (angle of the major axis, (-pi/2, pi/2])
//   t_mean   = sum q t / size
//   q_max    = largest q in the mask
//   out_params[e] = { size, cog_x, cog_y, length, width, psi, t_mean, q_max }   (8 x fp32)
//   n_pix == 0 or size <= 0 (or NaN)  ->  all eight parameters are 0.
//
// Everything between the fp32 inputs and the fp32 outputs is fp64, pixels in
// index order, centred second moments in a second pass.
//
// Shares no code with paper_1307_6489_b200/csrc. Parity status: pinned
// (tests/test_oracle_image_pins.py): a hand-worked 7-pixel camera
// (tests/golden/image7.json), closed forms (two pixels, lines, rotations,
// translations, charge scaling), eigenvalues of the covariance matrix by
// numpy.linalg.eigh, a vectorised numpy restatement of the cleaning, mutations.
#include <cmath>
#include <cstddef>
#include <cstdint>
#include <vector>

extern "C" {

// Returns 0 on success, 1 on a bad shape. out_mask may be null.
int rta_oracle_image_moments(const float* charge, const float* time, int64_t n_events,
                             int32_t n_pixels, const float* pix_x, const float* pix_y,
                             const int32_t* neighbors, float thr_picture, float thr_boundary,
                             int32_t* out_npix, float* out_params, uint8_t* out_mask) {
  if (n_events < 0 || n_pixels < 1) return 1;
  const int64_t P = n_pixels;
  std::vector<uint8_t> core(P), keep(P), mask(P);
  for (int64_t e = 0; e < n_events; ++e) {
    const float* q = charge + e * P;
    const float* t = time + e * P;
    for (int64_t p = 0; p < P; ++p) core[p] = q[p] >= thr_picture ? 1 : 0;
    for (int64_t p = 0; p < P; ++p) {
      bool any = false;
      for (int j = 0; j < 6; ++j) {
        const int32_t n = neighbors[p * 6 + j];
        if (n >= 0 && n < n_pixels && core[n]) any = true;
      }
      keep[p] = (core[p] && any) ? 1 : 0;
    }
    int32_t npix = 0;
    for (int64_t p = 0; p < P; ++p) {
      bool any = false;
      for (int j = 0; j < 6; ++j) {
        const int32_t n = neighbors[p * 6 + j];
        if (n >= 0 && n < n_pixels && keep[n]) any = true;
      }
      const bool edge = (q[p] >= thr_boundary) && any;
      mask[p] = (keep[p] || edge) ? 1 : 0;
      npix += mask[p];
      if (out_mask) out_mask[e * P + p] = mask[p];
    }
    double size = 0, sx = 0, sy = 0, st = 0;
    float qmax = 0.0f;
    bool first = true;
    for (int64_t p = 0; p < P; ++p) {
      if (!mask[p]) continue;
      const double w = (double)q[p];
      size += w;
      sx += w * (double)pix_x[p];
      sy += w * (double)pix_y[p];
      st += w * (double)t[p];
      if (first || q[p] > qmax) qmax = q[p];
      first = false;
    }
    out_npix[e] = npix;
    float* o = out_params + e * 8;
    if (npix == 0 || !(size > 0.0)) {
      for (int i = 0; i < 8; ++i) o[i] = 0.0f;
      continue;
    }
    const double cx = sx / size, cy = sy / size;
    double sxx = 0, syy = 0, sxy = 0;
    for (int64_t p = 0; p < P; ++p) {
      if (!mask[p]) continue;
      const double w = (double)q[p];
      const double dx = (double)pix_x[p] - cx, dy = (double)pix_y[p] - cy;
      sxx += w * dx * dx;
      syy += w * dy * dy;
      sxy += w * dx * dy;
    }
    sxx /= size;
    syy /= size;
    sxy /= size;
    const double d = sxx - syy;
    const double z = std::sqrt(d * d + 4.0 * sxy * sxy);
    const double l2 = 0.5 * (sxx + syy + z);
    double w2 = 0.5 * (sxx + syy - z);
    if (w2 < 0.0) w2 = 0.0;
    o[0] = (float)size;
    o[1] = (float)cx;
    o[2] = (float)cy;
    o[3] = (float)std::sqrt(l2);
    o[4] = (float)std::sqrt(w2);
    o[5] = (float)(0.5 * std::atan2(2.0 * sxy, d));
    o[6] = (float)(st / size);
    o[7] = qmax;
  }
  return 0;
}

}  // extern "C"
