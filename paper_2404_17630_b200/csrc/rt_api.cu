// The C ABI of include/rt.h: argument checking, marshalling and stream-ordered copies.
// All arithmetic of the method lives in rt_chem.cu / rt_transport.cu (per subcycle) and
// rt_setup.cu (per mesh).
#include <math.h>
#include <stdarg.h>
#include <string.h>
#include <algorithm>
#include <new>
#include <vector>
#include "rt_internal.cuh"

void rt_prof_begin(rt_ctx *c, int cls) {
  if (!c->prof_on) return;
  if (c->prof_used * 2 >= c->prof_ev.size()) {
    cudaEvent_t a, b;
    cudaEventCreate(&a); cudaEventCreate(&b);
    c->prof_ev.push_back(a); c->prof_ev.push_back(b);
    c->prof_cls.push_back(cls);
  }
  c->prof_cls[c->prof_used] = cls;
  cudaEventRecord(c->prof_ev[2 * c->prof_used], c->stream);
}
void rt_prof_end(rt_ctx *c) {
  if (!c->prof_on) return;
  cudaEventRecord(c->prof_ev[2 * c->prof_used + 1], c->stream);
  c->prof_used++;
}

int rt_fail(rt_ctx *c, int code, const char *fmt, ...) {
  if (c) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(c->err, sizeof(c->err), fmt, ap);
    va_end(ap);
  }
  return code;
}

extern "C" {

int rt_create(rt_ctx **out, int device, void *cuda_stream) {
  if (!out) return RT_EINVAL;
  *out = nullptr;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return RT_ECUDA;
  rt_ctx *c = new (std::nothrow) rt_ctx();
  if (!c) return RT_ENOMEM;
  c->device = 0; c->stream = 0; c->err[0] = 0; c->C = c->F = c->NR = 0; c->G = 0; c->nghost = 0; c->ws = nullptr;
  c->ws_bytes = 0; c->have_mesh = c->have_state = false; c->nsrc = 0; c->nsub_done = 0; c->launches = 0;
  c->prof_on = false; c->prof_used = 0; c->dbg_tl = nullptr; c->has_active = false;
  memset(&c->par, 0, sizeof(c->par)); memset(&c->lay, 0, sizeof(c->lay)); memset(&c->tun, 0, sizeof(c->tun));
  c->device = device;
  c->stream = (cudaStream_t)cuda_stream;
  if (cudaSetDevice(device) != cudaSuccess) { delete c; return RT_ECUDA; }
  *out = c;
  return RT_OK;
}

void rt_destroy(rt_ctx *c) {
  if (!c) return;
  for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
  delete c;
}

int rt_set_tuning(rt_ctx *c, const rt_tuning *t) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  rt_tuning z;
  memset(&z, 0, sizeof z);
  if (!t) t = &z;
  if (t->tile_cells != 0 && (t->tile_cells < RT_MIN_TILE || t->tile_cells > 1024))
    return rt_fail(c, RT_EINVAL, "tuning.tile_cells must be 0 or in [%d, 1024]", RT_MIN_TILE);
  if (t->tile_faces < -1 || t->tile_faces > RT_TILE_LIMIT) return rt_fail(c, RT_EINVAL, "tuning.tile_faces out of range");
  if (t->tile_blocks < 0 || t->tile_blocks > 8) return rt_fail(c, RT_EINVAL, "tuning.tile_blocks must be in [0, 8]");
  if (t->flux_threads < 0 || t->flux_threads > 256 || t->grad_threads < 0 || t->grad_threads > 256)
    return rt_fail(c, RT_EINVAL, "tuning.*_threads must be in [0, 256]");
  for (int k = 0; k < 6; k++)
    if (t->chem_caps[k] < 0) return rt_fail(c, RT_EINVAL, "tuning.chem_caps must be >= 0");
  c->tun = *t;
  return RT_OK;
}

int rt_profile(rt_ctx *c, int enable) {
  if (!c) return RT_EINVAL;
  c->prof_on = enable != 0;
  if (enable) c->prof_used = 0;
  return RT_OK;
}

int rt_profile_read(rt_ctx *c, double *ms, int64_t *count) {
  if (!c || !ms || !count) return RT_EINVAL;
  RT_CUDA(c, cudaStreamSynchronize(c->stream));
  for (int k = 0; k < RT_K_NCLS; k++) { ms[k] = 0.0; count[k] = 0; }
  for (size_t i = 0; i < c->prof_used; i++) {
    float t = 0.f;
    RT_CUDA(c, cudaEventElapsedTime(&t, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]));
    ms[c->prof_cls[i]] += t;
    count[c->prof_cls[i]]++;
  }
  c->prof_used = 0;
  return RT_OK;
}

const char *rt_last_error(const rt_ctx *c) { return c ? c->err : "null context"; }

int64_t rt_kernel_launches(const rt_ctx *c) { return c ? c->launches : 0; }

int rt_tile_info(const rt_ctx *c, int64_t *out) {
  if (!c || !out) return RT_EINVAL;
  if (!c->have_mesh) return RT_ESTATE;
  out[0] = c->TC; out[1] = c->T; out[2] = c->smax; out[3] = c->ninc;
  out[4] = c->hmax; out[5] = c->nhalo; out[6] = c->bmax; out[7] = c->blob_words;
  out[8] = c->omax; out[9] = c->fmax;
  out[10] = (int64_t)rt_smem_grad(c->TC, c->G, c->smax, c->hmax, c->bstride);
  out[11] = (int64_t)rt_smem_flux(c->TC, c->G, c->omax, c->fmax, c->bstride);
  out[12] = c->nFA; out[13] = c->omaxA; out[14] = c->fmaxA;
  out[15] = (int64_t)rt_smem_flux(c->TC, c->G, c->omaxA, c->fmaxA, c->bstride);
  return RT_OK;
}

size_t rt_workspace_bytes(int64_t ncell, int64_t nface, int ngroup, int flags) {
  if (ncell < 1 || nface < 1 || ngroup < 1 || ngroup > RT_MAXG || ncell > 0x7fffffffLL || nface > 0x7fffffffLL) return 0;
  return rt_make_layout(ncell, nface, ngroup, flags).total;
}

int rt_mesh_upload(rt_ctx *c, const rt_mesh *m, void *ws, size_t bytes) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  c->have_mesh = c->have_state = false;
  if (!m || !ws) return rt_fail(c, RT_EINVAL, "null mesh or workspace");
  if (m->ncell < 1 || m->nface < 1 || m->ncell > 0x7fffffffLL || m->nface > 0x7fffffffLL)
    return rt_fail(c, RT_EINVAL, "ncell/nface out of range");
  if (m->ngroup < 1 || m->ngroup > RT_MAXG) return rt_fail(c, RT_EINVAL, "ngroup must be in [1, %d]", RT_MAXG);
  if (!m->volume || !m->centroid || !m->area || !m->normal || !m->fcentroid || !m->left || !m->right)
    return rt_fail(c, RT_EINVAL, "null mesh array");
  if (m->nghost < 0 || m->nghost > 64 || (m->nghost > 0 && !m->ghost_state))
    return rt_fail(c, RT_EINVAL, "nghost must be in [0, 64] with ghost_state set");
  if (((uintptr_t)ws & 255) != 0) return rt_fail(c, RT_EINVAL, "workspace must be 256-byte aligned");
  for (int a = 0; a < 3; a++)
    if (!(m->box[a] > 0.0)) return rt_fail(c, RT_EINVAL, "box side must be positive");
  RT_CUDA(c, cudaSetDevice(c->device));
  c->C = m->ncell; c->F = m->nface; c->G = m->ngroup; c->nghost = m->nghost;
  for (int a = 0; a < 3; a++) { c->box[a] = m->box[a]; c->per[a] = m->periodic[a] != 0; }
  {  // mixed precision's length unit: the power of two next above the mean cell size
    int e;
    frexp(cbrt(m->box[0] * m->box[1] * m->box[2] / (double)m->ncell), &e);
    c->l0 = ldexp(1.0, e);
  }
  // the layout the caller's workspace was sized for: with room for every face's flux if it is that large
  const int devflag = m->mem_kind == RT_MEM_DEVICE ? RT_WS_DEVICE_MESH : 0;
  c->lay = rt_make_layout(c->C, c->F, c->G, devflag | RT_WS_ALL_FACES_CROSS);
  if (bytes < c->lay.total) c->lay = rt_make_layout(c->C, c->F, c->G, devflag);
  if (bytes < c->lay.total)
    return rt_fail(c, RT_ENOMEM, "workspace has %zu bytes, rt_workspace_bytes says %zu", bytes, c->lay.total);
  c->ws = (char *)ws;
  c->ws_bytes = bytes;
  int rc = rt_setup_mesh(c, m);
  if (rc != RT_OK) return rc;
  if ((rc = rt_transport_configure(c)) != RT_OK) return rc;
  c->have_mesh = true;
  return RT_OK;
}

// copy `rows` rows of C doubles (caller's order, host or device) into dst in the internal order
// dst[p*stride + r] = src[r][perm[p]]
static int put_rows(rt_ctx *c, const double *src, int mem_kind, double *dst, int rows, int stride, double *stage) {
  const size_t n = (size_t)rows * c->C;
  if (mem_kind == RT_MEM_HOST) {
    RT_CUDA(c, cudaMemcpyAsync(stage, src, n * 8, cudaMemcpyHostToDevice, c->stream));
    src = stage;
  }
  return rt_launch_permute_in(c, src, dst, rows, stride);
}

int rt_state_init(rt_ctx *c, const rt_params *p, const rt_state *s0, const rt_sources *src) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  if (!c->have_mesh) return rt_fail(c, RT_ESTATE, "rt_state_init needs rt_mesh_upload first");
  if (!p || !s0) return rt_fail(c, RT_EINVAL, "null params or state");
  if (p->ngroup != c->G) return rt_fail(c, RT_EINVAL, "params.ngroup %d != mesh.ngroup %d", p->ngroup, c->G);
  if (p->chem_mode < RT_CHEM_NONE || p->chem_mode > RT_CHEM_HHE_THERMAL) return rt_fail(c, RT_EINVAL, "bad chem_mode");
  if (!(p->ctilde > 0.0)) return rt_fail(c, RT_EINVAL, "ctilde must be positive");
  if (p->order < 1 || p->order > 2) return rt_fail(c, RT_EINVAL, "order must be 1 or 2");
  if (!s0->N || !s0->F) return rt_fail(c, RT_EINVAL, "state needs N and F");
  const bool chem = p->chem_mode >= RT_CHEM_H_ISOTHERMAL;
  if (chem && (!s0->xHII || !s0->xHeII || !s0->xHeIII || !s0->eth || !s0->nH))
    return rt_fail(c, RT_EINVAL, "chemistry needs xHII, xHeII, xHeIII, eth, nH");
  if (chem && (!(p->f_accept > 0.0) || !(p->f_target > 0.0) || p->max_substeps < 1))
    return rt_fail(c, RT_EINVAL, "chemistry needs f_accept, f_target > 0 and max_substeps >= 1");
  if (p->chem_mode == RT_CHEM_FIXED_OPACITY && !p->kappa) return rt_fail(c, RT_EINVAL, "FIXED_OPACITY needs kappa");
  if (p->mixed != 0 && p->mixed != 1) return rt_fail(c, RT_EINVAL, "mixed must be 0 or 1");
  const int nsrc = src ? src->nsrc : 0;
  if (nsrc < 0 || nsrc > 65536 || (nsrc > 0 && (!src->cell || !src->rate)))
    return rt_fail(c, RT_EINVAL, "nsrc must be in [0, 65536] with cell and rate set");
  for (int k = 0; k < nsrc; k++)
    if (src->cell[k] < 0 || src->cell[k] >= c->C) return rt_fail(c, RT_EINVAL, "source cell out of range");
  if (nsrc > 1) {  // the cells must be distinct: one source slot per cell (a duplicate would inject less than it books)
    std::vector<int32_t> seen(src->cell, src->cell + nsrc);
    std::sort(seen.begin(), seen.end());
    for (int k = 1; k < nsrc; k++)
      if (seen[k] == seen[k - 1]) return rt_fail(c, RT_EINVAL, "source cell %d is listed twice: sum its rates first", seen[k]);
  }
  RT_CUDA(c, cudaSetDevice(c->device));
  c->par = *p;
  c->par.kappa = nullptr;
  const rt_layout &l = c->lay;
  const int G = c->G;
  const int64_t C = c->C;
  double *stage = rt_ptr<double>(c, l.grad);  // 12 G C doubles: free between steps
  double *Ua = rt_ptr<double>(c, l.Ua);
  int rc;
  // N (G,C) and F (G,3,C) -> U[C][G][4]
  for (int g = 0; g < G; g++) {
    if ((rc = put_rows(c, s0->N + (size_t)g * C, s0->mem_kind, Ua + 4 * g, 1, 4 * G, stage))) return rc;
    if ((rc = put_rows(c, s0->F + (size_t)3 * g * C, s0->mem_kind, Ua + 4 * g + 1, 3, 4 * G, stage + C))) return rc;
    stage += 4 * C;
  }
  stage = rt_ptr<double>(c, l.grad) + (size_t)4 * G * C;
  const double *xs[5] = {s0->xHII, s0->xHeII, s0->xHeIII, s0->eth, s0->nH};
  const size_t xo[5] = {l.xHII, l.xHeII, l.xHeIII, l.eth, l.nH};
  for (int k = 0; k < 5; k++) {
    if (xs[k]) { if ((rc = put_rows(c, xs[k], s0->mem_kind, rt_ptr<double>(c, xo[k]), 1, 1, stage + (size_t)k * C))) return rc; }
    else RT_CUDA(c, cudaMemsetAsync(rt_ptr<double>(c, xo[k]), 0, 8 * C, c->stream));
  }
  if (p->chem_mode == RT_CHEM_FIXED_OPACITY) {
    if ((rc = put_rows(c, p->kappa, p->kappa_mem_kind, rt_ptr<double>(c, l.kappa), 1, 1, stage + (size_t)5 * C))) return rc;
  }
  // sources
  c->nsrc = nsrc;
  for (int g = 0; g < RT_MAXG; g++) { c->src_total[g] = 0.0; c->injected[g][0] = c->injected[g][1] = 0.0; }
  int32_t *cell_dev = rt_ptr<int32_t>(c, l.Ub);  // free until the first step
  if (nsrc > 0) {
    RT_CUDA(c, cudaMemcpyAsync(cell_dev, src->cell, 4 * (size_t)nsrc, cudaMemcpyHostToDevice, c->stream));
    RT_CUDA(c, cudaMemcpyAsync(rt_ptr<double>(c, l.srcrate), src->rate, 8 * (size_t)nsrc * G, cudaMemcpyHostToDevice, c->stream));
    for (int g = 0; g < G; g++) {
      double s = 0.0, cc = 0.0;
      for (int k = 0; k < nsrc; k++) {
        const double x = src->rate[(size_t)g * nsrc + k], t = s + x;
        cc += fabs(s) >= fabs(x) ? (s - t) + x : (x - t) + s;
        s = t;
      }
      c->src_total[g] = s + cc;
    }
  }
  c->src_cell.assign(src && nsrc > 0 ? src->cell : nullptr, src && nsrc > 0 ? src->cell + nsrc : nullptr);
  c->src_rate.assign(src && nsrc > 0 ? src->rate : nullptr, src && nsrc > 0 ? src->rate + (size_t)nsrc * G : nullptr);
  c->has_active = false;  // every cell active until rt_set_active says otherwise
  c->phase_next = 0;
  rt_launch_init_sources(c, cell_dev, nsrc);
  RT_CUDA(c, cudaMemsetAsync(rt_ptr<rt_dev_ledger>(c, l.led), 0, sizeof(rt_dev_ledger), c->stream));
  c->nsub_done = 0;
  RT_CUDA(c, cudaStreamSynchronize(c->stream));
  RT_CUDA(c, cudaGetLastError());
  c->have_state = true;
  return RT_OK;
}

int rt_set_active(rt_ctx *c, int mem_kind, const uint8_t *active) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  if (!c->have_state) return rt_fail(c, RT_ESTATE, "rt_set_active needs rt_state_init first");
  RT_CUDA(c, cudaSetDevice(c->device));
  const int G = c->G, nsrc = c->nsrc;
  std::vector<uint8_t> src_on((size_t)(nsrc > 0 ? nsrc : 0), 1);
  c->has_active = active != nullptr;
  if (active) {
    const uint8_t *dev = active;
    uint8_t *stage = rt_ptr<uint8_t>(c, c->lay.grad);  // 12 G C doubles: free between steps
    if (mem_kind == RT_MEM_HOST) {
      RT_CUDA(c, cudaMemcpyAsync(stage, active, (size_t)c->C, cudaMemcpyHostToDevice, c->stream));
      dev = stage;
      for (int k = 0; k < nsrc; k++) src_on[k] = (active[c->src_cell[k]] & 3) == 1;  // (a ghost's source is its owner's)
    } else {
      for (int k = 0; k < nsrc; k++)  // (a handful of one-byte copies: the source cells' flags)
        RT_CUDA(c, cudaMemcpyAsync(&src_on[k], active + c->src_cell[k], 1, cudaMemcpyDeviceToHost, c->stream));
    }
    int rc = rt_launch_active(c, dev);
    if (rc != RT_OK) return rc;
    RT_CUDA(c, cudaStreamSynchronize(c->stream));
    RT_CUDA(c, cudaGetLastError());
    if (mem_kind != RT_MEM_HOST)
      for (int k = 0; k < nsrc; k++) src_on[k] = (src_on[k] & 3) == 1;
  }
  // photons per unit time the active sources inject (the ledger's `injected` advances by dt times this)
  for (int g = 0; g < G; g++) {
    double s = 0.0, cc = 0.0;
    for (int k = 0; k < nsrc; k++) {
      if (!src_on[k]) continue;
      const double x = c->src_rate[(size_t)g * nsrc + k], t = s + x;
      cc += fabs(s) >= fabs(x) ? (s - t) + x : (x - t) + s;
      s = t;
    }
    c->src_total[g] = s + cc;
  }
  return RT_OK;
}

int rt_step_phase(rt_ctx *c, double dt, int phase) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  if (!c->have_state) return rt_fail(c, RT_ESTATE, "rt_step_phase needs rt_state_init first");
  if (!(dt > 0.0)) return rt_fail(c, RT_EINVAL, "dt must be positive");
  const int last = c->par.heun ? RT_PHASE_FLUX2 : RT_PHASE_FLUX1;
  if (phase < 0 || phase > last) return rt_fail(c, RT_EINVAL, "phase must be in [0, %d]", last);
  if (phase != c->phase_next)
    return rt_fail(c, RT_ESTATE, "phase %d out of order: phase %d of this subcycle comes next", phase, c->phase_next);
  RT_CUDA(c, cudaSetDevice(c->device));
  const int rc = rt_launch_phase(c, dt, phase);
  if (rc == RT_OK) c->phase_next = phase == last ? 0 : phase + 1;
  return rc;
}

static int halo_field(rt_ctx *c, int what, void **field, int *row_bytes) {
  const rt_layout &l = c->lay;
  if (what == RT_HALO_U) {  // the buffer the next gradient / flux phase reads: U^n, or U^1 in the second Heun stage
    const bool second = c->par.heun && c->phase_next >= RT_PHASE_GRAD2;
    *field = rt_ptr<double>(c, second ? l.Ub : l.Ua);
    *row_bytes = 32 * c->G;
  } else if (what == RT_HALO_GRAD) {
    *field = rt_ptr<double>(c, l.grad);
    *row_bytes = (c->par.mixed ? 48 : 96) * c->G;
  } else return rt_fail(c, RT_EINVAL, "what must be RT_HALO_U or RT_HALO_GRAD");
  return RT_OK;
}

static int halo_call(rt_ctx *c, bool pack, int what, int64_t n, const int32_t *cells_dev, void *buf_dev, const char *name) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  if (!c->have_state) return rt_fail(c, RT_ESTATE, "%s needs rt_state_init first", name);
  if (n < 0 || (n > 0 && (!cells_dev || !buf_dev))) return rt_fail(c, RT_EINVAL, "%s: null pointer or negative count", name);
  if (((uintptr_t)buf_dev & 15) != 0) return rt_fail(c, RT_EINVAL, "%s: the buffer must be 16-byte aligned", name);
  RT_CUDA(c, cudaSetDevice(c->device));
  void *field = nullptr;
  int row_bytes = 0;
  const int rc = halo_field(c, what, &field, &row_bytes);
  if (rc != RT_OK) return rc;
  return rt_launch_halo(c, pack, field, row_bytes, n, cells_dev, buf_dev);
}

int rt_halo_pack(rt_ctx *c, int what, int64_t n, const int32_t *cells_dev, void *buf_dev) {
  return halo_call(c, true, what, n, cells_dev, buf_dev, "rt_halo_pack");
}
int rt_halo_unpack(rt_ctx *c, int what, int64_t n, const int32_t *cells_dev, const void *buf_dev) {
  return halo_call(c, false, what, n, cells_dev, (void *)buf_dev, "rt_halo_unpack");
}

int rt_halo_row_bytes(const rt_ctx *c, int what) {
  if (!c || !c->have_state) return RT_EINVAL;
  return what == RT_HALO_U ? 32 * c->G : what == RT_HALO_GRAD ? (c->par.mixed ? 48 : 96) * c->G : RT_EINVAL;
}

int rt_step(rt_ctx *c, double dt, int nsub) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  if (!c->have_state) return rt_fail(c, RT_ESTATE, "rt_step needs rt_state_init first");
  if (c->phase_next != 0) return rt_fail(c, RT_ESTATE, "rt_step inside a subcycle begun with rt_step_phase (phase %d comes next)", c->phase_next);
  if (!(dt > 0.0) || nsub < 0) return rt_fail(c, RT_EINVAL, "dt must be positive and nsub >= 0");
  RT_CUDA(c, cudaSetDevice(c->device));
  for (int s = 0; s < nsub; s++) {
    int rc = rt_launch_step(c, dt);
    if (rc != RT_OK) return rc;
  }
  return RT_OK;
}

// dst[r][perm[p]] = src[p*stride + r]
static int get_rows(rt_ctx *c, const double *src, double *dst, int mem_kind, int rows, int stride, double *stage) {
  const size_t n = (size_t)rows * c->C;
  if (mem_kind == RT_MEM_HOST) {
    rt_launch_permute_out(c, src, stage, rows, stride);
    RT_CUDA(c, cudaMemcpyAsync(dst, stage, n * 8, cudaMemcpyDeviceToHost, c->stream));
    return RT_OK;
  }
  return rt_launch_permute_out(c, src, dst, rows, stride);
}

int rt_download(rt_ctx *c, rt_state *out, rt_ledger *led) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  if (!c->have_state) return rt_fail(c, RT_ESTATE, "rt_download needs rt_state_init first");
  RT_CUDA(c, cudaSetDevice(c->device));
  const rt_layout &l = c->lay;
  const int G = c->G;
  const int64_t C = c->C;
  int rc;
  if (out) {
    double *stage = rt_ptr<double>(c, l.grad);
    const double *Ua = rt_ptr<double>(c, l.Ua);
    for (int g = 0; g < G; g++) {
      if (out->N && (rc = get_rows(c, Ua + 4 * g, out->N + (size_t)g * C, out->mem_kind, 1, 4 * G, stage))) return rc;
      if (out->F && (rc = get_rows(c, Ua + 4 * g + 1, out->F + (size_t)3 * g * C, out->mem_kind, 3, 4 * G, stage + C)))
        return rc;
      stage += 4 * C;
    }
    double *xs[4] = {out->xHII, out->xHeII, out->xHeIII, out->eth};
    const size_t xo[4] = {l.xHII, l.xHeII, l.xHeIII, l.eth};
    for (int k = 0; k < 4; k++)
      if (xs[k] && (rc = get_rows(c, rt_ptr<double>(c, xo[k]), xs[k], out->mem_kind, 1, 1, stage + (size_t)k * C))) return rc;
  }
  rt_dev_ledger h;
  if (led) {
    rt_launch_stored(c);
    RT_CUDA(c, cudaMemcpyAsync(&h, rt_ptr<rt_dev_ledger>(c, l.led), sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  }
  RT_CUDA(c, cudaStreamSynchronize(c->stream));
  RT_CUDA(c, cudaGetLastError());
  if (led) {
    memset(led, 0, sizeof(*led));
    for (int g = 0; g < G; g++) {
      led->absorbed[g] = h.acc[0][g][0] + h.acc[0][g][1];
      led->outflow[g] = h.acc[1][g][0] + h.acc[1][g][1];
      led->inflow_bc[g] = h.acc[2][g][0] + h.acc[2][g][1];
      led->floor_added[g] = h.acc[3][g][0] + h.acc[3][g][1];
      led->stored[g] = h.acc[4][g][0];
      led->injected[g] = c->injected[g][0] + c->injected[g][1];
    }
    led->substeps_total = (int64_t)h.substeps_total;
    led->substeps_max = (int64_t)h.substeps_max;
    led->cells_hit_cap = (int64_t)h.cells_hit_cap;
    led->nsub_done = c->nsub_done;
  }
  return RT_OK;
}

int rt_debug_tile_timeline(rt_ctx *c, double dt, int64_t ntile_max, uint64_t *out) {
  if (!c || !out) return RT_EINVAL;
  c->err[0] = 0;
  if (!c->have_state) return rt_fail(c, RT_ESTATE, "rt_debug_tile_timeline needs rt_state_init first");
  if (!(dt > 0.0) || ntile_max < c->T) return rt_fail(c, RT_EINVAL, "dt must be positive and out must hold 8 words for each of the %lld tiles", (long long)c->T);
  RT_CUDA(c, cudaSetDevice(c->device));
  unsigned long long *buf = nullptr;
  RT_CUDA(c, cudaMalloc(&buf, 64 * (size_t)c->T));  // (a debug call: allocates outside the caller's workspace)
  RT_CUDA(c, cudaMemsetAsync(buf, 0, 64 * (size_t)c->T, c->stream));
  c->dbg_tl = buf;
  const int rc = rt_launch_step(c, dt);
  c->dbg_tl = nullptr;
  cudaError_t e = cudaMemcpyAsync(out, buf, 64 * (size_t)c->T, cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  cudaFree(buf);
  if (e != cudaSuccess) return rt_fail(c, RT_ECUDA, "timeline copy: %s", cudaGetErrorString(e));
  return rc;
}

__global__ void k_tile_of_cell(int64_t C, int TC, const int32_t *__restrict__ perm, int32_t *__restrict__ out) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p < C) out[perm[p]] = (int32_t)(p / TC);
}

int rt_debug_tiles(rt_ctx *c, int mem_kind, int32_t *tile_of_cell, int32_t *tile_desc) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  if (!c->have_mesh) return rt_fail(c, RT_ESTATE, "rt_debug_tiles needs rt_mesh_upload first");
  RT_CUDA(c, cudaSetDevice(c->device));
  const rt_layout &l = c->lay;
  if (tile_of_cell) {
    int32_t *dst = tile_of_cell, *tmp = nullptr;
    if (mem_kind == RT_MEM_HOST) { RT_CUDA(c, cudaMalloc(&tmp, 4 * (size_t)c->C)); dst = tmp; }  // (a debug call)
    k_tile_of_cell<<<(unsigned)((c->C + 255) / 256), 256, 0, c->stream>>>(c->C, c->TC, rt_ptr<int32_t>(c, l.perm), dst);
    cudaError_t e = cudaSuccess;
    if (tmp) e = cudaMemcpyAsync(tile_of_cell, tmp, 4 * (size_t)c->C, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (tmp) cudaFree(tmp);
    if (e != cudaSuccess) return rt_fail(c, RT_ECUDA, "rt_debug_tiles: %s", cudaGetErrorString(e));
  }
  if (tile_desc) {
    std::vector<rt_tile> d((size_t)c->T);
    std::vector<int32_t> list((size_t)c->T);
    RT_CUDA(c, cudaMemcpyAsync(d.data(), rt_ptr<rt_tile>(c, l.tiles), sizeof(rt_tile) * (size_t)c->T, cudaMemcpyDeviceToHost, c->stream));
    RT_CUDA(c, cudaMemcpyAsync(list.data(), rt_ptr<int32_t>(c, l.tlistF), 4 * (size_t)c->T, cudaMemcpyDeviceToHost, c->stream));
    RT_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int64_t t = 0; t < c->T; t++) {
      tile_desc[4 * t] = d[t].nown; tile_desc[4 * t + 1] = d[t].nh - d[t].nb;
      tile_desc[4 * t + 2] = rt_blob_words(c->TC, d[t].nhf, d[t].nown, d[t].nh, d[t].ninc, d[t].nout);
      tile_desc[4 * t + 3] = 1;
    }
    for (int64_t k = 0; k < c->nFA; k++) tile_desc[4 * (int64_t)list[k] + 3] = 0;  // class-A tiles come first in the flux list
  }
  RT_CUDA(c, cudaGetLastError());
  return RT_OK;
}

int rt_debug_gradients(rt_ctx *c, int mem_kind, double *gN, double *gF) {
  if (!c) return RT_EINVAL;
  c->err[0] = 0;
  if (!c->have_state) return rt_fail(c, RT_ESTATE, "rt_debug_gradients needs rt_state_init first");
  if (!gN || !gF) return rt_fail(c, RT_EINVAL, "null output");
  RT_CUDA(c, cudaSetDevice(c->device));
  const rt_layout &l = c->lay;
  const int64_t C = c->C;
  const int mixed = c->par.mixed;  // (always the fp64 gradients, in the caller's units: the mixed mode's are l0-scaled floats)
  c->par.mixed = 0;
  rt_launch_gradients(c, rt_ptr<double>(c, l.Ua));
  c->par.mixed = mixed;
  double *grad = rt_ptr<double>(c, l.grad);
  double *stage = rt_ptr<double>(c, l.Ub);  // 4 G C doubles, free between steps; used 3 and 9 rows at a time
  int rc;
  for (int g = 0; g < c->G; g++) {
    if ((rc = get_rows(c, grad + 12 * g, gN + (size_t)3 * g * C, mem_kind, 3, 12 * c->G, stage))) return rc;
    RT_CUDA(c, cudaStreamSynchronize(c->stream));
    // 9 rows do not fit a 4-row stage when G == 1: go 3 rows at a time
    for (int q = 0; q < 3; q++) {
      if ((rc = get_rows(c, grad + 12 * g + 3 + 3 * q, gF + (size_t)(9 * g + 3 * q) * C, mem_kind, 3, 12 * c->G, stage)))
        return rc;
      RT_CUDA(c, cudaStreamSynchronize(c->stream));
    }
  }
  RT_CUDA(c, cudaGetLastError());
  return RT_OK;
}

}  // extern "C"
