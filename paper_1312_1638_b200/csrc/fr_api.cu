// C ABI of the FR library (include/fr.h): context management, constant uploads, RHS and RK4 drivers.
#include <cstdio>
#include <cstring>
#include <exception>
#include <new>
#include <string>
#include <type_traits>
#include <vector>

#include "fr_dev.hpp"
#include "fr_host.hpp"
#include "fr_element.hpp"
#include "fr_hex_tma.hpp"
#include "fr_tensor.hpp"

using namespace fr;

struct fr_ctx {
  MeshInput mesh;
  RefOps ops;
  MeshConsts mc;
  fr_disc_desc disc{};
  bool ready = false;
  bool use_tensor = false;
  bool host_only = false;
  DevConsts dc{};
  WorkLayout wl{};
  TensorPlan tp{};
  std::vector<void *> dev_allocs;
  mutable std::string err;
};

static thread_local std::string g_setup_err;

namespace {

int fail(const fr_ctx *c, int code, const std::string &msg) {
  if (c) c->err = msg; else g_setup_err = msg;
  return code;
}

void free_dev(fr_ctx *c) {
  for (void *p : c->dev_allocs) cudaFree(p);
  c->dev_allocs.clear();
}

template <typename T>
cudaError_t upload(fr_ctx *c, const std::vector<T> &h, const T **dptr) {
  *dptr = nullptr;
  if (h.empty()) return cudaSuccess;
  void *d = nullptr;
  cudaError_t e = cudaMalloc(&d, h.size() * sizeof(T));
  if (e != cudaSuccess) return e;
  c->dev_allocs.push_back(d);
  e = cudaMemcpy(d, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
  *dptr = (const T *)d;
  return e;
}

int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

}  // namespace

extern "C" {

int fr_setup_mesh(fr_ctx **out, const fr_mesh_desc *m) {
  if (!out) return fail(nullptr, FR_EINVAL, "fr_setup_mesh: out is NULL");
  *out = nullptr;
  if (!m) return fail(nullptr, FR_EINVAL, "fr_setup_mesh: mesh is NULL");
  try {
    const int nd_expected = (m->etype == FR_HEX) ? 3 : 2;
    if (m->etype != FR_QUAD && m->etype != FR_TRI && m->etype != FR_HEX) return fail(nullptr, FR_EINVAL, "unknown element type");
    if (m->ndims != nd_expected) return fail(nullptr, FR_EINVAL, "ndims does not match the element type");
    if (m->n_elems <= 0 || m->n_elems > 2000000000LL) return fail(nullptr, FR_EINVAL, "n_elems out of range");
    if (m->p_g < 1 || m->p_g > 8) return fail(nullptr, FR_EINVAL, "p_g out of range [1,8]");
    if (!m->nodes) return fail(nullptr, FR_EINVAL, "nodes is NULL");
    if ((m->n_ifaces > 0 && (!m->ifaces || !m->shifts)) || (m->n_bfaces > 0 && (!m->bfaces || !m->bcs)) || m->n_ifaces < 0 || m->n_bfaces < 0)
      return fail(nullptr, FR_EINVAL, "interface / boundary arrays missing");
    int m1 = m->p_g + 1;
    int64_t Nn = (m->etype == FR_TRI) ? m1 * (m1 + 1) / 2 : (m->etype == FR_QUAD ? m1 * m1 : m1 * m1 * m1);
    fr_ctx *c = new fr_ctx();
    c->mesh.nd = m->ndims; c->mesh.etype = m->etype; c->mesh.p_g = m->p_g; c->mesh.Nel = m->n_elems;
    c->mesh.nodes.assign(m->nodes, m->nodes + (size_t)m->n_elems * Nn * m->ndims);
    if (m->n_ifaces) {
      c->mesh.ifaces.assign(m->ifaces, m->ifaces + (size_t)m->n_ifaces * 4);
      c->mesh.shifts.assign(m->shifts, m->shifts + (size_t)m->n_ifaces * m->ndims);
    }
    if (m->n_bfaces) c->mesh.bfaces.assign(m->bfaces, m->bfaces + (size_t)m->n_bfaces * 3);
    if (m->n_bcs > 0 && m->bcs) c->mesh.bcs.assign(m->bcs, m->bcs + m->n_bcs);
    for (auto &b : c->mesh.bcs)
      if (b.kind < FR_BC_SUP_INFLOW || b.kind > FR_BC_NOSLIP_WALL) { delete c; return fail(nullptr, FR_EINVAL, "unknown boundary condition kind"); }
    *out = c;
    return FR_OK;
  } catch (const std::bad_alloc &) {
    return fail(nullptr, FR_ENOMEM, "out of host memory");
  } catch (const std::exception &ex) {
    return fail(nullptr, FR_EINVAL, ex.what());
  }
}

int fr_setup_operators(fr_ctx *c, const fr_disc_desc *d) {
  if (!c) return fail(nullptr, FR_EINVAL, "fr_setup_operators: ctx is NULL");
  if (!d) return fail(c, FR_EINVAL, "fr_setup_operators: disc is NULL");
  if (d->system != FR_EULER && d->system != FR_NAVIER_STOKES) return fail(c, FR_EINVAL, "unknown system");
  if (d->precision != FR_F32 && d->precision != FR_F64) return fail(c, FR_EINVAL, "unknown precision");
  if (!(d->gamma > 1.0)) return fail(c, FR_EINVAL, "gamma must be > 1");
  if (d->system == FR_NAVIER_STOKES && (!(d->mu >= 0.0) || !(d->Pr > 0.0))) return fail(c, FR_EINVAL, "mu >= 0 and Pr > 0 required");
  try {
    c->ready = false;
    free_dev(c);
    build_ref_ops(c->mesh.etype, d->p, c->mesh.p_g, c->ops);
    const int64_t lane = FR_BLK;  // rows start on 128-byte boundaries (north_star) and hold whole element blocks (fp_row)
    const int64_t ld = align_up(c->mesh.Nel, lane);
    std::string err;
    c->host_only = (d->flags & FR_FLAG_HOST_ONLY) != 0;
    // hexahedra on the TMA-pipelined kernels keep every internal array element-blocked (fr_dev.hpp: fp_row)
    const bool blk = !c->host_only && !(d->flags & FR_FLAG_FORCE_GENERIC) && c->ops.etype == FR_HEX &&
                     hex_tma_supported(c->ops.n, d->precision == FR_F64);
    int rc = build_mesh_consts(c->mesh, c->ops, ld, blk ? FR_BLK : 0, c->mc, err);
    if (rc != FR_OK) return fail(c, rc, err);
    c->disc = *d;
    const RefOps &o = c->ops;
    const MeshConsts &mc = c->mc;
    DevConsts &dc = c->dc;
    dc = DevConsts();
    dc.nd = o.nd; dc.NV = o.nd + 2; dc.Nu = o.Nu; dc.Nf = o.Nf; dc.n = o.n; dc.nfp = o.nfp; dc.etype = o.etype;
    dc.Nel = mc.Nel; dc.ld = ld; dc.npairs = mc.npairs; dc.nbnd = mc.nbnd;
    dc.ns = d->system == FR_NAVIER_STOKES; dc.f64 = d->precision == FR_F64;
    dc.staged = (d->flags & FR_FLAG_FORCE_GENERIC) != 0;
    dc.ph = Phys{d->gamma, d->mu, d->Pr, d->ldg_beta, d->ldg_tau};
    dc.dev = -1;
    if (c->host_only) { c->use_tensor = false; c->wl = WorkLayout(); c->ready = true; return FR_OK; }
    cudaError_t e = cudaGetDevice(&dc.dev);
    if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    dc.blk = blk;
    auto reblock = [&](const auto &src, int rows) {  // [rows][ld] -> [ld / FR_BLK][rows][FR_BLK]
      typename std::decay<decltype(src)>::type dst(src.size());
      for (int64_t b = 0; b < ld / FR_BLK; ++b)
        for (int r = 0; r < rows; ++r)
          std::memcpy(&dst[((size_t)b * rows + r) * FR_BLK], &src[(size_t)r * ld + (size_t)b * FR_BLK], FR_BLK * sizeof(src[0]));
      return dst;
    };
#define UP(vec, field) if (e == cudaSuccess) e = upload(c, vec, &dc.field)
    UP(o.M[0], M0); UP(o.M[3], M3); UP(o.M[6], M6); UP(o.M46, M46); UP(o.M132, M132);
    dc.hM0 = o.M[0].data(); dc.hM3 = o.M[3].data(); dc.hM6 = o.M[6].data(); dc.hM46 = o.M46.data(); dc.hM132 = o.M132.data();
    dc.affine = mc.affine;
    dc.aff = dc.blk && mc.affine;
    if (dc.aff) {  // affine hexahedra: one point of S and 1/J per element; the tensor maps broadcast it (fr_tma.cuh: encode_blk)
      const int nn = o.nd * o.nd;
      std::vector<double> s_el((size_t)nn * ld), r_el((size_t)ld);
      for (int cc = 0; cc < nn; ++cc) std::memcpy(&s_el[(size_t)cc * ld], &mc.smat[(size_t)cc * o.Nu * ld], ld * sizeof(double));
      std::memcpy(r_el.data(), mc.rcpj.data(), ld * sizeof(double));
      UP(reblock(s_el, nn), smat); UP(reblock(r_el, 1), rcpj);
    } else if (dc.blk) { UP(reblock(mc.smat, o.nd * o.nd * o.Nu), smat); UP(reblock(mc.rcpj, o.Nu), rcpj); }
    else { UP(mc.smat, smat); UP(mc.rcpj, rcpj); }
    UP(mc.pLs, pLs); UP(mc.pLe, pLe); UP(mc.pRs, pRs); UP(mc.pRe, pRe);
    UP(mc.pn, pn); UP(mc.pJnL, pJnL); UP(mc.pJnR, pJnR);
    UP(mc.bs, bs); UP(mc.be, be); UP(mc.bbc, bbc); UP(mc.bn, bn); UP(mc.bJn, bJn);
    // element-centric flux-point tables of the fused hexahedral gradient kernel (own normals, boundary ids)
    const bool want_tma = !(d->flags & FR_FLAG_FORCE_GENERIC) && o.etype == FR_HEX && dc.ns && hex_tma_supported(o.n, dc.f64);
    if (want_tma) {
      UP(reblock(mc.fp_n, o.nd * o.Nf), fp_n);
      if (mc.nbnd) { UP(reblock(mc.fp_pe, o.Nf), fp_pe); }
    }
    const bool want_el = dc.ns && element_fused_supported(dc);  // fused triangle kernels
    if (want_el) { UP(mc.fp_n, fp_n); if (mc.nbnd) { UP(mc.fp_pe, fp_pe); } }
    if (want_tma) {
      // faces whose G^f enters the common flux: L sides weigh 1/2 + beta, R sides 1/2 - beta (Eq 27), boundaries always
      std::vector<uint8_t> need((size_t)o.nfaces * ld, 0);
      for (int f = 0; f < o.nfaces; ++f)
        for (int64_t el = 0; el < mc.Nel; ++el) {
          const size_t i0 = (size_t)(f * o.nfp) * ld + el;
          const bool bnd = mc.fp_pe[i0] < 0, rside = mc.fp_Jn[i0] < 0;
          need[(size_t)f * ld + el] = bnd || (rside ? 0.5 - d->ldg_beta : 0.5 + d->ldg_beta) != 0.0;
        }
      UP(need, face_need);
    }
#undef UP
    std::vector<BcDev> bcs(c->mesh.bcs.size());
    for (size_t i = 0; i < bcs.size(); ++i) {
      const fr_bc_desc &b = c->mesh.bcs[i];
      bcs[i] = BcDev{b.kind, b.rho, {b.v[0], b.v[1], b.v[2]}, b.p, b.cpTw};
    }
    dc.nbcs = (int)bcs.size();
    if (e == cudaSuccess) e = upload(c, bcs, &dc.bcs);
    if (e != cudaSuccess) { free_dev(c); return fail(c, FR_ECUDA, std::string("constant upload: ") + cudaGetErrorString(e)); }

    // workspace layout
    const int64_t esz = dc.f64 ? 8 : 4;
    const int64_t state = (int64_t)o.Nu * dc.NV * ld * esz;
    WorkLayout &w = c->wl;
    int64_t off = 0;
    auto take = [&](int64_t bytes) { int64_t o2 = off; off = align_up(off + bytes, 256); return o2; };
    c->use_tensor = false;
    if (!(d->flags & FR_FLAG_FORCE_GENERIC) && tensor_supported(dc) && !element_fused_supported(dc)) {
      e = tensor_plan(dc, o, mc, c->tp, c->dev_allocs);
      if (e != cudaSuccess) { free_dev(c); return fail(c, FR_ECUDA, std::string("tensor plan: ") + cudaGetErrorString(e)); }
      c->use_tensor = true;
      w.uf = take(c->tp.work_bytes);
      w.cf = w.qu = w.qf = w.uf;
    } else {
      w.uf = take((int64_t)o.Nf * dc.NV * ld * 8);
      w.cf = dc.ns ? take((int64_t)o.Nf * dc.NV * ld * 8) : 0;
      w.qu = take((int64_t)o.nd * o.Nu * dc.NV * ld * 8);
      w.qf = dc.ns ? take((int64_t)o.nd * o.Nf * dc.NV * ld * 8) : 0;
    }
    w.rk_k = take(state); w.rk_tmp = take(state); w.rk_acc = take(state);
    w.total = off;
    c->ready = true;
    return FR_OK;
  } catch (const std::bad_alloc &) {
    return fail(c, FR_ENOMEM, "out of host memory");
  } catch (const std::exception &ex) {
    return fail(c, FR_EINVAL, ex.what());
  }
}

#define FR_NEED_READY(c, ret) \
  if (!(c)) return ret;      \
  if (!(c)->ready) { (c)->err = "fr_setup_operators has not completed"; return ret; }

int64_t fr_num_solution_points(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->ops.Nu; }
int64_t fr_num_flux_points(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->ops.Nf; }
int64_t fr_num_vars(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->dc.NV; }
int64_t fr_num_pairs(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->mc.npairs; }
int64_t fr_leading_dim(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->dc.ld; }
int64_t fr_state_bytes(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return (int64_t)c->ops.Nu * c->dc.NV * c->dc.ld * (c->dc.f64 ? 8 : 4); }
int64_t fr_workspace_bytes(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->wl.total; }
int64_t fr_rhs_kernel_launches(const fr_ctx *c) {
  FR_NEED_READY(c, FR_EINVAL)
  return c->use_tensor ? tensor_rhs_launches(c->dc) : generic_rhs_launches(c->dc);
}

int fr_solution_point_coords(const fr_ctx *c, double *xyz) {
  FR_NEED_READY(c, FR_EINVAL)
  if (!xyz) return fail(c, FR_EINVAL, "xyz_host is NULL");
  std::memcpy(xyz, c->mc.xu.data(), c->mc.xu.size() * sizeof(double));
  return FR_OK;
}

int fr_operator_dims(const fr_ctx *c, int id, int64_t *rows, int64_t *cols) {
  FR_NEED_READY(c, FR_EINVAL)
  if (id < 0 || id > 6 || !rows || !cols) return fail(c, FR_EINVAL, "operator id out of range or NULL output");
  *rows = c->ops.rows[id]; *cols = c->ops.cols[id];
  return FR_OK;
}

int fr_get_operator(const fr_ctx *c, int id, double *buf) {
  FR_NEED_READY(c, FR_EINVAL)
  if (id < 0 || id > 6 || !buf) return fail(c, FR_EINVAL, "operator id out of range or NULL buffer");
  std::memcpy(buf, c->ops.M[id].data(), c->ops.M[id].size() * sizeof(double));
  return FR_OK;
}

int fr_get_pairs(const fr_ctx *c, int32_t *pairs, double *normals, double *jn) {
  FR_NEED_READY(c, FR_EINVAL)
  const MeshConsts &m = c->mc;
  const int nd = c->ops.nd;
  for (int64_t i = 0; i < m.npairs; ++i) {
    if (pairs) { pairs[4 * i] = m.pLs[i]; pairs[4 * i + 1] = m.pLe[i]; pairs[4 * i + 2] = m.pRs[i]; pairs[4 * i + 3] = m.pRe[i]; }
    if (normals) for (int n = 0; n < nd; ++n) normals[i * nd + n] = m.pn[(size_t)n * m.npairs + i];
    if (jn) { jn[2 * i] = m.pJnL[i]; jn[2 * i + 1] = m.pJnR[i]; }
  }
  return FR_OK;
}

int fr_get_metrics(const fr_ctx *c, double *smat, double *rcpj) {
  FR_NEED_READY(c, FR_EINVAL)
  if (smat) std::memcpy(smat, c->mc.smat.data(), c->mc.smat.size() * sizeof(double));
  if (rcpj) std::memcpy(rcpj, c->mc.rcpj.data(), c->mc.rcpj.size() * sizeof(double));
  return FR_OK;
}

static int rhs_impl(fr_ctx *c, const void *u, void *rhs, void *work, void *stream, Prof *prof) {
  FR_NEED_READY(c, FR_EINVAL)
  if (!u || !rhs || !work) return fail(c, FR_EINVAL, "fr_rhs: NULL device pointer");
  if (u == rhs) return fail(c, FR_EINVAL, "fr_rhs: rhs must not alias u");
  if (c->host_only) return fail(c, FR_EINVAL, "fr_rhs: context was set up with FR_FLAG_HOST_ONLY");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != c->dc.dev)
    return fail(c, FR_EINVAL, "fr_rhs: the current CUDA device is not the one fr_setup_operators uploaded the constants to");
  cudaStream_t s = (cudaStream_t)stream;
  cudaError_t e = c->use_tensor ? tensor_rhs(c->dc, c->tp, u, rhs, (char *)work + c->wl.uf, s, prof)
                                : generic_rhs(c->dc, c->wl, u, rhs, (char *)work, s, prof);
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_rhs launch: ") + cudaGetErrorString(e));
  return FR_OK;
}

int fr_rhs(fr_ctx *c, const void *u, void *rhs, void *work, void *stream) { return rhs_impl(c, u, rhs, work, stream, nullptr); }

int fr_rhs_profiled(fr_ctx *c, const void *u, void *rhs, void *work, void *stream, int max_kernels, int *n_kernels,
                    float *ms, char *names) {
  FR_NEED_READY(c, FR_EINVAL)
  if (!n_kernels || !ms || !names || max_kernels <= 0) return fail(c, FR_EINVAL, "fr_rhs_profiled: NULL output");
  Prof prof;
  prof.s = (cudaStream_t)stream;
  for (int i = 0; i <= Prof::MAXK; ++i) cudaEventCreate(&prof.ev[i]);
  int rc = rhs_impl(c, u, rhs, work, stream, &prof);
  prof.end();
  cudaError_t e = cudaStreamSynchronize(prof.s);
  int n = prof.n < max_kernels ? prof.n : max_kernels;
  for (int i = 0; i < n && e == cudaSuccess; ++i) {
    e = cudaEventElapsedTime(&ms[i], prof.ev[i], prof.ev[i + 1]);
    std::snprintf(names + 32 * i, 32, "%s", prof.names[i]);
  }
  *n_kernels = n;
  for (int i = 0; i <= Prof::MAXK; ++i) cudaEventDestroy(prof.ev[i]);
  if (rc != FR_OK) return rc;
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_rhs_profiled: ") + cudaGetErrorString(e));
  return FR_OK;
}

int fr_rk4_step(fr_ctx *c, void *u, double dt, void *work, void *stream) {
  FR_NEED_READY(c, FR_EINVAL)
  if (c->host_only) return fail(c, FR_EINVAL, "fr_rk4_step: context was set up with FR_FLAG_HOST_ONLY");
  if (!u || !work) return fail(c, FR_EINVAL, "fr_rk4_step: NULL device pointer");
  cudaStream_t s = (cudaStream_t)stream;
  char *wk = (char *)work;
  void *k = wk + c->wl.rk_k, *tmp = wk + c->wl.rk_tmp, *acc = wk + c->wl.rk_acc;
  const int64_t n = (int64_t)c->ops.Nu * c->dc.NV;  // rows of ld values; pad columns (e >= n_elems) are left untouched
  const bool f64 = c->dc.f64;
  int rc;
  cudaError_t e;
  // k1; tmp = u + dt/2 k1; acc = u + dt/6 k1
  if ((rc = fr_rhs(c, u, k, work, stream)) != FR_OK) return rc;
  e = rk_axpy2(f64, n, c->dc.ld, c->dc.Nel, u, k, dt / 2, tmp, dt / 6, acc, 0, s);
  // k2; tmp = u + dt/2 k2; acc += dt/3 k2
  if (e == cudaSuccess && (rc = fr_rhs(c, tmp, k, work, stream)) != FR_OK) return rc;
  if (e == cudaSuccess) e = rk_axpy2(f64, n, c->dc.ld, c->dc.Nel, u, k, dt / 2, tmp, dt / 3, acc, 1, s);
  // k3; tmp = u + dt k3; acc += dt/3 k3
  if (e == cudaSuccess && (rc = fr_rhs(c, tmp, k, work, stream)) != FR_OK) return rc;
  if (e == cudaSuccess) e = rk_axpy2(f64, n, c->dc.ld, c->dc.Nel, u, k, dt, tmp, dt / 3, acc, 1, s);
  // k4; u = acc + dt/6 k4
  if (e == cudaSuccess && (rc = fr_rhs(c, tmp, k, work, stream)) != FR_OK) return rc;
  if (e == cudaSuccess) e = rk_axpy2(f64, n, c->dc.ld, c->dc.Nel, u, k, 0.0, u, dt / 6, acc, 2, s);
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_rk4_step launch: ") + cudaGetErrorString(e));
  return FR_OK;
}

int fr_rhs_host(fr_ctx *c, const void *u_host, void *rhs_host, void *u_dev, void *rhs_dev, void *work, void *stream) {
  FR_NEED_READY(c, FR_EINVAL)
  if (!u_host || !rhs_host || !u_dev || !rhs_dev || !work) return fail(c, FR_EINVAL, "fr_rhs_host: NULL pointer");
  cudaStream_t s = (cudaStream_t)stream;
  const size_t bytes = (size_t)fr_state_bytes(c);
  cudaError_t e = cudaMemcpyAsync(u_dev, u_host, bytes, cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("H2D: ") + cudaGetErrorString(e));
  int rc = fr_rhs(c, u_dev, rhs_dev, work, stream);
  if (rc != FR_OK) return rc;
  e = cudaMemcpyAsync(rhs_host, rhs_dev, bytes, cudaMemcpyDeviceToHost, s);
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("D2H: ") + cudaGetErrorString(e));
  return FR_OK;
}

void fr_teardown(fr_ctx *c) {
  if (!c) return;
  free_dev(c);
  delete c;
}

const char *fr_last_error(const fr_ctx *c) { return c ? c->err.c_str() : g_setup_err.c_str(); }

}  // extern "C"
