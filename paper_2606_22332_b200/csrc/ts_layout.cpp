// S0 -- taxel-layout builder (host).  See include/ts.h for the contract and citations
// (P:178 probe = position + unit normal + radius; P:182 R_j = 0 fillers; P:72 regular planar
// grids; P:510 link filters).  Coordinates are evaluated in double and rounded to fp32 once.
#include "ts_internal.h"

#include <cmath>
#include <new>

namespace {
inline double dot3(const float* a, const float* b) {
  return (double)a[0] * b[0] + (double)a[1] * b[1] + (double)a[2] * b[2];
}
}  // namespace

extern "C" {

ts_status ts_layout_create(ts_layout** out) {
  if (!out) return TS_ERR_INVALID_ARG;
  ts_layout* l = new (std::nothrow) ts_layout();
  if (!l) return TS_ERR_OOM;
  *out = l;
  return TS_OK;
}

ts_status ts_layout_add_patch(ts_layout* lay, const ts_patch_desc* d) {
  if (!lay || !d || lay->finalized) return TS_ERR_INVALID_ARG;
  if (d->nu < 1 || d->nv < 1 || d->nu * d->nv > TS_MAX_PATCH_TAXELS) return TS_ERR_INVALID_ARG;
  if (d->marker_nu < 0 || d->marker_nv < 0 || d->marker_nu * d->marker_nv > TS_MAX_PATCH_TAXELS) return TS_ERR_INVALID_ARG;
  if ((d->marker_nu == 0) != (d->marker_nv == 0)) return TS_ERR_INVALID_ARG;
  if (!(d->radius > 0.0f) || !(d->size_u > 0.0f) || !(d->size_v > 0.0f) || d->link < 0) return TS_ERR_INVALID_ARG;
  double uu = dot3(d->u_axis, d->u_axis), vv = dot3(d->v_axis, d->v_axis), uv = dot3(d->u_axis, d->v_axis);
  // unit and orthogonal to 1e-5: the separable marker sums (ts_kernels.cu phase 5) rely on |r|^2 = du^2 + dv^2
  if (std::fabs(uu - 1.0) > 1e-5 || std::fabs(vv - 1.0) > 1e-5 || std::fabs(uv) > 1e-5) return TS_ERR_INVALID_ARG;
  const double ux = d->u_axis[0], uy = d->u_axis[1], uz = d->u_axis[2];
  const double vx = d->v_axis[0], vy = d->v_axis[1], vz = d->v_axis[2];
  const double n[3] = {uy * vz - uz * vy, uz * vx - ux * vz, ux * vy - uy * vx};
  lay->desc.push_back(*d);
  const int p = (int)lay->patch_start.size();
  const int t0 = (int)lay->radius.size();
  lay->patch_start.push_back(t0);
  lay->patch_nu.push_back(d->nu);
  lay->patch_nv.push_back(d->nv);
  lay->patch_link.push_back(d->link);
  lay->patch_eps.push_back((float)((double)d->size_u / d->nu));
  for (int iv = 0; iv < d->nv; ++iv)
    for (int iu = 0; iu < d->nu; ++iu) {
      const double su = ((iu + 0.5) / d->nu - 0.5) * (double)d->size_u;
      const double sv = ((iv + 0.5) / d->nv - 0.5) * (double)d->size_v;
      lay->pos.push_back((float)(d->origin[0] + su * ux + sv * vx));
      lay->pos.push_back((float)(d->origin[1] + su * uy + sv * vy));
      lay->pos.push_back((float)(d->origin[2] + su * uz + sv * vz));
      for (int a = 0; a < 3; ++a) lay->nrm.push_back((float)n[a]);
      lay->radius.push_back(d->radius);
      lay->radius_cfg.push_back(d->radius);
      lay->link.push_back(d->link);
      lay->patch.push_back(p);
    }
  lay->marker_start.push_back((int)lay->marker_patch.size());
  lay->marker_count.push_back(d->marker_nu * d->marker_nv);
  for (int iv = 0; iv < d->marker_nv; ++iv)
    for (int iu = 0; iu < d->marker_nu; ++iu) {
      const double su = ((iu + 0.5) / d->marker_nu - 0.5) * (double)d->size_u;
      const double sv = ((iv + 0.5) / d->marker_nv - 0.5) * (double)d->size_v;
      lay->marker_pos.push_back((float)(d->origin[0] + su * ux + sv * vx));
      lay->marker_pos.push_back((float)(d->origin[1] + su * uy + sv * vy));
      lay->marker_pos.push_back((float)(d->origin[2] + su * uz + sv * vz));
      for (int a = 0; a < 3; ++a) lay->marker_nrm.push_back((float)n[a]);
      lay->marker_patch.push_back(p);
    }
  return TS_OK;
}

ts_status ts_layout_filter_links(ts_layout* lay, const uint8_t* link_mask, int32_t n_links) {
  if (!lay || !link_mask || n_links < 1) return TS_ERR_INVALID_ARG;
  for (size_t t = 0; t < lay->radius_cfg.size(); ++t) {
    const int l = lay->link[t];
    if (l >= n_links) return TS_ERR_INVALID_ARG;
    lay->radius[t] = link_mask[l] ? lay->radius_cfg[t] : 0.0f;
  }
  return TS_OK;
}

ts_status ts_layout_finalize(ts_layout* lay, int32_t n_taxels) {
  if (!lay || lay->finalized) return TS_ERR_INVALID_ARG;
  const int used = (int)lay->radius_cfg.size();
  if (n_taxels < used || n_taxels < 1) return TS_ERR_INVALID_ARG;
  for (int t = used; t < n_taxels; ++t) {  // trailing fillers
    for (int a = 0; a < 3; ++a) lay->pos.push_back(0.0f);
    lay->nrm.push_back(0.0f); lay->nrm.push_back(0.0f); lay->nrm.push_back(1.0f);
    lay->radius.push_back(0.0f);
    lay->radius_cfg.push_back(0.0f);
    lay->link.push_back(0);
    lay->patch.push_back(-1);
  }
  lay->nbr.assign((size_t)n_taxels * 4, -1);
  for (size_t p = 0; p < lay->patch_start.size(); ++p) {
    const int s = lay->patch_start[p], nu = lay->patch_nu[p], nv = lay->patch_nv[p];
    for (int iv = 0; iv < nv; ++iv)
      for (int iu = 0; iu < nu; ++iu) {
        const int t = s + iv * nu + iu;
        int* nb = &lay->nbr[(size_t)t * 4];
        nb[0] = iu > 0 ? t - 1 : -1;
        nb[1] = iu < nu - 1 ? t + 1 : -1;
        nb[2] = iv > 0 ? t - nu : -1;
        nb[3] = iv < nv - 1 ? t + nu : -1;
      }
  }
  lay->n_taxels = n_taxels;
  lay->finalized = true;
  return TS_OK;
}

ts_status ts_layout_get(const ts_layout* lay, ts_layout_view* v) {
  if (!lay || !v || !lay->finalized) return TS_ERR_INVALID_ARG;
  v->n_taxels = lay->n_taxels;
  v->n_patches = (int32_t)lay->patch_start.size();
  v->n_markers = (int32_t)lay->marker_patch.size();
  v->pos = lay->pos.data(); v->nrm = lay->nrm.data(); v->radius = lay->radius.data();
  v->link = lay->link.data(); v->patch = lay->patch.data(); v->nbr = lay->nbr.data();
  v->patch_start = lay->patch_start.data(); v->patch_nu = lay->patch_nu.data(); v->patch_nv = lay->patch_nv.data();
  v->patch_link = lay->patch_link.data();
  v->marker_start = lay->marker_start.data(); v->marker_count = lay->marker_count.data();
  v->marker_pos = lay->marker_pos.data(); v->marker_nrm = lay->marker_nrm.data();
  v->marker_patch = lay->marker_patch.data();
  return TS_OK;
}

ts_status ts_layout_destroy(ts_layout* lay) {
  delete lay;
  return TS_OK;
}

}  // extern "C"
