// C ABI of the FR library (include/fr.h): context management, constant uploads, RHS and RK4 drivers.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <cstdint>
#include <exception>
#include <mutex>
#include <new>
#include <string>
#include <type_traits>
#include <vector>

#include "fr_dev.hpp"
#include "fr_host.hpp"
#include "fr_element.hpp"
#include "fr_hex_tma.hpp"
#include "fr_mixed.hpp"
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
  bool lean = false;  // FR_FLAG_LEAN: host tables released after upload
  DevConsts dc{};
  WorkLayout wl{};
  TensorPlan tp{};
  std::vector<void *> dev_allocs;
  mutable std::string err;
  // ---- mesh of several element types (fr_setup_mesh_mixed): one sub-context per part, cross-part tables here ----
  bool sub = false;                  // this context is a part of a mixed mesh
  std::vector<fr_ctx *> parts;       // owned
  std::vector<int32_t> mx_ifaces;    // [n][6]
  std::vector<double> mx_shifts;
  MixedPairs mx{};
  std::vector<int64_t> mx_soff;      // byte offset of every part in a state buffer
  std::vector<int64_t> mx_fpo;       // offset (doubles) of every part inside a flux-point region
  std::vector<int64_t> mx_qoff;      // byte offset of every part's Q array in the workspace
  int64_t mx_state = 0, mx_region = 0, mx_uf = 0, mx_cf = 0, mx_gf = 0;  // total state bytes; region size (doubles); region byte offsets
  ~fr_ctx() { for (fr_ctx *q : parts) delete q; }
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
  if (c->dc.map_cache) { hex_tma_cache_destroy(c->dc.map_cache); c->dc.map_cache = nullptr; }
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

int fr_setup_mesh_mixed(fr_ctx **out, const fr_mixed_mesh_desc *m) {
  if (!out) return fail(nullptr, FR_EINVAL, "fr_setup_mesh_mixed: out is NULL");
  *out = nullptr;
  if (!m) return fail(nullptr, FR_EINVAL, "fr_setup_mesh_mixed: mesh is NULL");
  if (m->ndims != 2) return fail(nullptr, FR_EUNSUPPORTED, "mixed meshes are two-dimensional (quadrilaterals and triangles)");
  if (m->n_parts < 1 || m->n_parts > 8 || !m->parts) return fail(nullptr, FR_EINVAL, "n_parts out of range [1,8]");
  if (m->n_ifaces < 0 || m->n_bfaces < 0 || (m->n_ifaces > 0 && (!m->ifaces || !m->shifts)) || (m->n_bfaces > 0 && (!m->bfaces || !m->bcs)))
    return fail(nullptr, FR_EINVAL, "interface / boundary arrays missing");
  fr_ctx *c = nullptr;
  try {
    c = new fr_ctx();
    c->mesh.nd = 2;
    for (int t = 0; t < m->n_parts; ++t) {
      const fr_mesh_part &pt = m->parts[t];
      if (pt.etype != FR_QUAD && pt.etype != FR_TRI) { delete c; return fail(nullptr, FR_EINVAL, "a part of a mixed mesh must hold quadrilaterals or triangles"); }
      // boundary faces of this part as a single-type list
      std::vector<int32_t> bf;
      for (int64_t b = 0; b < m->n_bfaces; ++b)
        if (m->bfaces[4 * b] == t) { bf.push_back(m->bfaces[4 * b + 1]); bf.push_back(m->bfaces[4 * b + 2]); bf.push_back(m->bfaces[4 * b + 3]); }
      fr_mesh_desc d1{};
      d1.ndims = 2; d1.etype = pt.etype; d1.p_g = pt.p_g; d1.n_bcs = m->n_bcs; d1.n_elems = pt.n_elems;
      d1.n_ifaces = 0; d1.n_bfaces = (int64_t)bf.size() / 3; d1.nodes = pt.nodes; d1.bfaces = bf.data(); d1.bcs = m->bcs;
      fr_ctx *q = nullptr;
      const int rc = fr_setup_mesh(&q, &d1);
      if (rc != FR_OK) { delete c; return rc; }  // text already in g_setup_err
      q->sub = true;
      c->parts.push_back(q);
    }
    for (int64_t f = 0; f < m->n_ifaces; ++f) {
      const int32_t *r = m->ifaces + 6 * f;
      if (r[0] < 0 || r[0] >= m->n_parts || r[3] < 0 || r[3] >= m->n_parts) { delete c; return fail(nullptr, FR_EINVAL, "interface record references a part out of range"); }
    }
    for (int64_t b = 0; b < m->n_bfaces; ++b)
      if (m->bfaces[4 * b] < 0 || m->bfaces[4 * b] >= m->n_parts) { delete c; return fail(nullptr, FR_EINVAL, "boundary face references a part out of range"); }
    c->mx_ifaces.assign(m->ifaces, m->ifaces + (size_t)m->n_ifaces * 6);
    c->mx_shifts.assign(m->shifts, m->shifts + (size_t)m->n_ifaces * 2);
    *out = c;
    return FR_OK;
  } catch (const std::bad_alloc &) {
    delete c;
    return fail(nullptr, FR_ENOMEM, "out of host memory");
  } catch (const std::exception &ex) {
    delete c;
    return fail(nullptr, FR_EINVAL, ex.what());
  }
}

static int setup_mixed(fr_ctx *c, const fr_disc_desc *d);

int fr_setup_operators(fr_ctx *c, const fr_disc_desc *d) {
  if (!c) return fail(nullptr, FR_EINVAL, "fr_setup_operators: ctx is NULL");
  if (!c->parts.empty()) return setup_mixed(c, d);
  if (!d) return fail(c, FR_EINVAL, "fr_setup_operators: disc is NULL");
  if (d->system != FR_EULER && d->system != FR_NAVIER_STOKES) return fail(c, FR_EINVAL, "unknown system");
  if (d->precision != FR_F32 && d->precision != FR_F64) return fail(c, FR_EINVAL, "unknown precision");
  if (!(d->gamma > 1.0)) return fail(c, FR_EINVAL, "gamma must be > 1");
  if (d->system == FR_NAVIER_STOKES && (!(d->mu >= 0.0) || !(d->Pr > 0.0))) return fail(c, FR_EINVAL, "mu >= 0 and Pr > 0 required");
  if (c->lean) return fail(c, FR_EINVAL, "fr_setup_operators: the context was set up with FR_FLAG_LEAN (host mesh released)");
  try {
    c->ready = false;
    free_dev(c);
    build_ref_ops(c->mesh.etype, d->p, c->mesh.p_g, d->correction, c->ops);
    const int64_t lane = FR_BLK;  // rows start on 128-byte boundaries (north_star) and hold whole element blocks (fp_row)
    const int64_t ld = align_up(c->mesh.Nel, lane);
    std::string err;
    c->host_only = (d->flags & FR_FLAG_HOST_ONLY) != 0;
    // hexahedra on the TMA-pipelined kernels keep every internal array element-blocked (fr_dev.hpp: fp_row)
    const bool blk = !c->host_only && !(d->flags & FR_FLAG_FORCE_GENERIC) && c->ops.etype == FR_HEX &&
                     hex_tma_supported(c->ops.n, d->precision == FR_F64);
    int rc = build_mesh_consts(c->mesh, c->ops, ld, blk ? FR_BLK : 0, c->mc, err, !c->sub);
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
    dc.force_el = c->sub;
    // the reference state (perturbation form, fr_physics.cuh) serves the fused kernel families; the staged sequence and the
    // line kernels of high-order quadrilaterals evaluate the plain formulas
    const bool fused = !dc.staged && (o.etype == FR_HEX ? blk : element_fused_supported(dc));
    const double zero3[3] = {0, 0, 0};
    dc.ph = make_phys(d->gamma, d->mu, d->Pr, d->ldg_beta, d->ldg_tau, fused ? d->rho_ref : 0.0, fused ? d->v_ref : zero3, fused ? d->p_ref : 0.0);
    dc.dev = -1;
    if (c->host_only) { c->use_tensor = false; c->wl = WorkLayout(); c->ready = true; return FR_OK; }
    cudaError_t e = cudaGetDevice(&dc.dev);
    if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    dc.blk = blk;
    dc.map_cache = blk ? hex_tma_cache_create() : nullptr;
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
    // The hexahedral TMA path keeps its metric terms, normals and J n in the STORAGE precision (single precision halves
    // their traffic too; with a reference state their rounding multiplies deviation-sized fluxes only, fr_physics.cuh).
    const bool f32tab = dc.blk && !dc.f64;
    auto up_t = [&](const std::vector<double> &v, const double **dst) {  // upload as double, or as float behind the same pointer
      if (!f32tab) return upload(c, v, dst);
      std::vector<float> f(v.begin(), v.end());
      const float *p = nullptr;
      cudaError_t er = upload(c, f, &p);
      *dst = (const double *)(const void *)p;
      return er;
    };
#define UPT(vec, field) if (e == cudaSuccess) e = up_t(vec, &dc.field)
    if (dc.aff) {  // affine hexahedra: one point of S and 1/J per element; the tensor maps broadcast it (fr_tma.cuh: encode_blk)
      const int nn = o.nd * o.nd;
      std::vector<double> s_el((size_t)nn * ld), r_el((size_t)ld);
      for (int cc = 0; cc < nn; ++cc) std::memcpy(&s_el[(size_t)cc * ld], &mc.smat[(size_t)cc * o.Nu * ld], ld * sizeof(double));
      std::memcpy(r_el.data(), mc.rcpj.data(), ld * sizeof(double));
      UPT(reblock(s_el, nn), smat); UPT(reblock(r_el, 1), rcpj);
    } else if (dc.blk) { UPT(reblock(mc.smat, o.nd * o.nd * o.Nu), smat); UPT(reblock(mc.rcpj, o.Nu), rcpj); }
    else { UP(mc.smat, smat); UP(mc.rcpj, rcpj); }
    UP(mc.pLs, pLs); UP(mc.pLe, pLe); UP(mc.pRs, pRs); UP(mc.pRe, pRe);
    if (dc.aff) {
      // affine hexahedra: normal and J n of a flux point are those of its face (first flux point of the face); per-face tables
      // replace the per-pair ones (fr_dev.hpp: pf_n): 4 nd (nd + 1) words per element instead of (nd + 2) N_f / 2
      const int nf = o.nfaces;
      std::vector<double> fn((size_t)o.nd * nf * ld, 0.0), fj((size_t)nf * ld, 0.0);
      for (int f = 0; f < nf; ++f)
        for (int64_t el = 0; el < mc.Nel; ++el) {
          const int sg = f * o.nfp;
          for (int n = 0; n < o.nd; ++n) fn[((size_t)n * nf + f) * ld + el] = mc.fp_n[((size_t)n * o.Nf + sg) * ld + el];
          fj[(size_t)f * ld + el] = std::fabs(mc.fp_Jn[(size_t)sg * ld + el]);  // (the sign bit marks R sides)
        }
      UPT(fn, pf_n); UPT(fj, pf_Jn);
    } else {
      UPT(mc.pn, pn); UPT(mc.pJnL, pJnL); UPT(mc.pJnR, pJnR);
    }
    UP(mc.bs, bs); UP(mc.be, be); UP(mc.bbc, bbc); UP(mc.bn, bn); UP(mc.bJn, bJn);
    // element-centric flux-point tables of the fused hexahedral gradient kernel (own normals, boundary ids)
    const bool want_tma = !(d->flags & FR_FLAG_FORCE_GENERIC) && o.etype == FR_HEX && dc.ns && hex_tma_supported(o.n, dc.f64);
    if (want_tma) {
      UPT(reblock(mc.fp_n, o.nd * o.Nf), fp_n);
      // partner of every flux point as an offset into the element-blocked U^f array (row sigma * N_V of N_f * N_V rows)
      std::vector<int64_t> poff((size_t)o.Nf * ld, 0);
      for (int sg = 0; sg < o.Nf; ++sg)
        for (int64_t el = 0; el < mc.Nel; ++el) {
          const size_t i0 = (size_t)sg * ld + el;
          const int32_t pe = mc.fp_pe[i0];
          poff[i0] = pe < 0 ? (int64_t)pe : (int64_t)fp_row(true, ld, o.Nf * dc.NV, mc.fp_ps[i0] * dc.NV, pe);
        }
      UP(reblock(poff, o.Nf), fp_poff);
    }
    const bool want_el = dc.ns && element_fused_supported(dc);  // fused triangle / quadrilateral kernels
    if (want_el) { UP(mc.fp_n, fp_n); if (mc.nbnd) { UP(mc.fp_pe, fp_pe); } }
    if (want_el && !c->sub) {
      // the fused 2-D gradient kernel forms the common solution itself (Eq 7, 25): partner of every flux point as an offset
      // into U^f [N_f][N_V][ld], and on which side of its interface the flux point lies (1 = L, 2 = R, 3 = boundary)
      std::vector<int64_t> poff((size_t)o.Nf * ld, 0);
      std::vector<uint8_t> code((size_t)o.Nf * ld, 0);
      for (int sg = 0; sg < o.Nf; ++sg)
        for (int64_t el = 0; el < mc.Nel; ++el) {
          const size_t i0 = (size_t)sg * ld + el;
          const int32_t pe = mc.fp_pe[i0];
          poff[i0] = pe < 0 ? 0 : (int64_t)mc.fp_ps[i0] * dc.NV * ld + pe;
          code[i0] = pe < 0 ? 3 : (mc.fp_Jn[i0] < 0 ? 2 : 1);
        }
      UP(poff, fp_poff);
      UP(code, face_code);
    }
    if (want_tma) {
      // faces that carry an LDG weight (jump of Eq 9 and G^f of Eq 27): L sides weigh 1/2 + beta, R sides 1/2 - beta
      std::vector<uint8_t> code((size_t)o.nfaces * ld, 0);
      for (int f = 0; f < o.nfaces; ++f)
        for (int64_t el = 0; el < mc.Nel; ++el) {
          const size_t i0 = (size_t)(f * o.nfp) * ld + el;
          const bool bnd = mc.fp_pe[i0] < 0, rside = mc.fp_Jn[i0] < 0;
          const double wgt = rside ? 0.5 - d->ldg_beta : 0.5 + d->ldg_beta;
          code[(size_t)f * ld + el] = bnd ? 3 : (wgt == 0.0 ? 0 : (rside ? 2 : 1));
        }
      UP(code, face_code);
    }
#undef UP
#undef UPT
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
    w.partials = take((int64_t)RK_MAX_PARTIALS * 8);
    w.reg0 = off; w.reg_stride = align_up(state, 256);
    w.total = w.reg0 + 3 * w.reg_stride;
    if (d->flags & FR_FLAG_LEAN) {
      auto drop = [](auto &v) { typename std::decay<decltype(v)>::type().swap(v); };
      MeshConsts &m = c->mc;
      drop(m.smat); drop(m.rcpj); drop(m.pLs); drop(m.pLe); drop(m.pRs); drop(m.pRe); drop(m.pn); drop(m.pJnL); drop(m.pJnR);
      drop(m.bs); drop(m.be); drop(m.bbc); drop(m.bn); drop(m.bJn); drop(m.fp_pe); drop(m.fp_ps); drop(m.fp_n); drop(m.fp_Jn);
      drop(c->mesh.nodes); drop(c->mesh.ifaces); drop(c->mesh.shifts); drop(c->mesh.bfaces);
      c->lean = true;
    }
    c->ready = true;
    return FR_OK;
  } catch (const std::bad_alloc &) {
    return fail(c, FR_ENOMEM, "out of host memory");
  } catch (const std::exception &ex) {
    return fail(c, FR_EINVAL, ex.what());
  }
}

// ---- mesh of several element types: parts set up one by one, then the cross-part lookup table ----
static int setup_mixed(fr_ctx *c, const fr_disc_desc *d) {
  if (!d) return fail(c, FR_EINVAL, "fr_setup_operators: disc is NULL");
  if (d->flags & (FR_FLAG_FORCE_GENERIC | FR_FLAG_HOST_ONLY | FR_FLAG_LEAN)) return fail(c, FR_EUNSUPPORTED, "mixed meshes: flags are not supported");
  if (d->p < 1 || d->p > 4) return fail(c, FR_EUNSUPPORTED, "mixed meshes run the fused element kernels: 1 <= p <= 4");
  try {
    c->ready = false;
    free_dev(c);
    const int np_ = (int)c->parts.size(), nd = 2, NV = 4;
    for (fr_ctx *q : c->parts) {
      const int rc = fr_setup_operators(q, d);
      if (rc != FR_OK) return fail(c, rc, "part: " + q->err);
      if (!element_fused_supported(q->dc)) return fail(c, FR_EUNSUPPORTED, "mixed meshes need the fused element kernels for every part");
    }
    c->disc = *d;
    c->dc = c->parts[0]->dc;  // N_V, physics, precision, device
    // layout of a state buffer and of the flux-point regions
    const int64_t esz = c->dc.f64 ? 8 : 4;
    c->mx_soff.assign(np_, 0); c->mx_fpo.assign(np_, 0); c->mx_qoff.assign(np_, 0);
    int64_t so = 0, fo = 0;
    for (int t = 0; t < np_; ++t) {
      const DevConsts &q = c->parts[t]->dc;
      c->mx_soff[t] = so; so = align_up(so + (int64_t)q.Nu * NV * q.ld * esz, 256);
      c->mx_fpo[t] = fo; fo = align_up(fo + (int64_t)q.Nf * NV * q.ld, 32);
    }
    c->mx_state = so; c->mx_region = fo;
    // cross-part pairing by physical coordinates (:182, A11)
    struct Pr { int64_t oL, oR; int32_t vL, vR; double n0, n1, jL, jR; };
    const int64_t nif = (int64_t)c->mx_ifaces.size() / 6;
    std::vector<Pr> pairs;
    std::vector<std::vector<int32_t>> cover(np_);
    for (int t = 0; t < np_; ++t) cover[t].assign((size_t)c->parts[t]->ops.Nf * c->parts[t]->mc.Nel, 0);
    int64_t unmatched = 0;
    for (int64_t f = 0; f < nif; ++f) {
      const int32_t *r = &c->mx_ifaces[6 * f];
      const fr_ctx *L = c->parts[r[0]], *R = c->parts[r[3]];
      const int nfp = L->ops.nfp;
      if (R->ops.nfp != nfp) return fail(c, FR_EMESH, "the two sides of an interface have different numbers of flux points");
      const int64_t eL = r[1], eR = r[4];
      if (eL < 0 || eL >= L->mc.Nel || eR < 0 || eR >= R->mc.Nel || r[2] < 0 || r[2] >= L->ops.nfaces || r[5] < 0 || r[5] >= R->ops.nfaces)
        return fail(c, FR_EINVAL, "interface list references an element or face out of range");
      auto xL = [&](int s, int n) { return L->mc.xf[((size_t)s * L->mc.Nel + eL) * nd + n]; };
      auto xR = [&](int s, int n) { return R->mc.xf[((size_t)s * R->mc.Nel + eR) * nd + n] + c->mx_shifts[(size_t)f * nd + n]; };
      double h2 = 0;
      for (int n = 0; n < nd; ++n) { const double dd = xL(r[2] * nfp, n) - xL(r[2] * nfp + nfp - 1, n); h2 += dd * dd; }
      const double tol2 = 1e-18 * (h2 > 0 ? h2 : 1.0) + 1e-24;
      unsigned long long used = 0;
      for (int k = 0; k < nfp; ++k) {
        const int sL = r[2] * nfp + k;
        int best = -1;
        double bd = 1e300;
        for (int mm = 0; mm < nfp; ++mm) {
          double d2 = 0;
          for (int n = 0; n < nd; ++n) { const double dd = xL(sL, n) - xR(r[5] * nfp + mm, n); d2 += dd * dd; }
          if (d2 < bd) { bd = d2; best = mm; }
        }
        if (!(bd <= tol2) || ((used >> best) & 1ull)) ++unmatched;
        used |= 1ull << best;
        const int sR = r[5] * nfp + best;
        const int64_t ldL = L->dc.ld, ldR = R->dc.ld;
        Pr pr;
        pr.oL = c->mx_fpo[r[0]] + (int64_t)sL * NV * ldL + eL; pr.vL = (int32_t)ldL;
        pr.oR = c->mx_fpo[r[3]] + (int64_t)sR * NV * ldR + eR; pr.vR = (int32_t)ldR;
        pr.n0 = L->mc.fp_n[((size_t)0 * L->ops.Nf + sL) * ldL + eL]; pr.n1 = L->mc.fp_n[((size_t)1 * L->ops.Nf + sL) * ldL + eL];
        pr.jL = L->mc.fp_Jn[(size_t)sL * ldL + eL]; pr.jR = R->mc.fp_Jn[(size_t)sR * ldR + eR];
        pairs.push_back(pr);
        cover[r[0]][(size_t)sL * L->mc.Nel + eL]++; cover[r[3]][(size_t)sR * R->mc.Nel + eR]++;
      }
    }
    if (unmatched) return fail(c, FR_EMESH, "unmatched flux-point pairs: " + std::to_string(unmatched));
    for (int t = 0; t < np_; ++t) {
      const fr_ctx *q = c->parts[t];
      for (int64_t i = 0; i < q->mc.nbnd; ++i) cover[t][(size_t)q->mc.bs[i] * q->mc.Nel + q->mc.be[i]]++;
      for (auto v : cover[t]) if (v != 1) return fail(c, FR_EMESH, "flux points not covered exactly once by interfaces + boundary faces");
    }
    std::sort(pairs.begin(), pairs.end(), [](const Pr &a, const Pr &b) { return a.oL < b.oL; });  // coalesced L side (:693)
    const int64_t n = (int64_t)pairs.size();
    std::vector<int64_t> oL(n), oR(n);
    std::vector<int32_t> vL(n), vR(n);
    std::vector<double> nrm(2 * (size_t)n), jL(n), jR(n);
    for (int64_t i = 0; i < n; ++i) {
      oL[i] = pairs[i].oL; oR[i] = pairs[i].oR; vL[i] = pairs[i].vL; vR[i] = pairs[i].vR;
      nrm[i] = pairs[i].n0; nrm[(size_t)n + i] = pairs[i].n1; jL[i] = pairs[i].jL; jR[i] = pairs[i].jR;
    }
    cudaError_t e = cudaSuccess;
    c->mx = MixedPairs();
    c->mx.n = n;
    e = upload(c, oL, &c->mx.oL);
    if (e == cudaSuccess) e = upload(c, oR, &c->mx.oR);
    if (e == cudaSuccess) e = upload(c, vL, &c->mx.vL);
    if (e == cudaSuccess) e = upload(c, vR, &c->mx.vR);
    if (e == cudaSuccess) e = upload(c, nrm, &c->mx.nrm);
    if (e == cudaSuccess) e = upload(c, jL, &c->mx.jL);
    if (e == cudaSuccess) e = upload(c, jR, &c->mx.jR);
    if (e != cudaSuccess) { free_dev(c); return fail(c, FR_ECUDA, std::string("constant upload: ") + cudaGetErrorString(e)); }
    for (fr_ctx *q : c->parts) std::vector<double>().swap(q->mc.xf);
    // workspace: U^f (-> D~), C^f, G^f regions, Q of every part, stepper registers
    int64_t off = 0;
    auto take = [&](int64_t bytes) { int64_t o2 = off; off = align_up(off + bytes, 256); return o2; };
    c->mx_uf = take(c->mx_region * 8);
    c->mx_cf = c->dc.ns ? take(c->mx_region * 8) : 0;
    c->mx_gf = c->dc.ns ? take(c->mx_region * 8) : 0;
    for (int t = 0; t < np_; ++t) {
      const DevConsts &q = c->parts[t]->dc;
      c->mx_qoff[t] = c->dc.ns ? take((int64_t)nd * q.Nu * NV * q.ld * 8) : 0;
    }
    WorkLayout &w = c->wl;
    w = WorkLayout();
    w.partials = take((int64_t)RK_MAX_PARTIALS * 8);
    w.reg0 = off; w.reg_stride = align_up(c->mx_state, 256);
    w.total = w.reg0 + 3 * w.reg_stride;
    c->ready = true;
    return FR_OK;
  } catch (const std::bad_alloc &) {
    return fail(c, FR_ENOMEM, "out of host memory");
  } catch (const std::exception &ex) {
    return fail(c, FR_EINVAL, ex.what());
  }
}

// rhs of a mixed mesh: the fused element kernels part by part, the interface kernels over all flux-point pairs at once
static cudaError_t mixed_rhs(fr_ctx *c, const void *u, void *rhs, char *work, cudaStream_t s, Prof *prof) {
  const int np_ = (int)c->parts.size();
  double *uf = (double *)(work + c->mx_uf), *cf = (double *)(work + c->mx_cf), *gf = (double *)(work + c->mx_gf);
  const bool ns = c->dc.ns;
  cudaError_t e = cudaSuccess;
  auto up = [&](int t) { return (const void *)((const char *)u + c->mx_soff[t]); };
  FR_MARK(prof, "el_interp");
  for (int t = 0; t < np_ && e == cudaSuccess; ++t) e = element_interp(c->parts[t]->dc, up(t), uf + c->mx_fpo[t], s);
  if (e != cudaSuccess) return e;
  if (ns) {
    FR_MARK(prof, "common_sol");
    mixed_common_sol(c->mx, c->dc.ph, uf, cf, s);
    for (int t = 0; t < np_; ++t)
      if (c->parts[t]->dc.nbnd) launch_common_sol(c->parts[t]->dc, uf + c->mx_fpo[t], cf + c->mx_fpo[t], s);
    FR_MARK(prof, "el_gradface");
    for (int t = 0; t < np_ && e == cudaSuccess; ++t)
      e = element_gradface(c->parts[t]->dc, up(t), cf + c->mx_fpo[t], uf + c->mx_fpo[t], (double *)(work + c->mx_qoff[t]), gf + c->mx_fpo[t], s);
    if (e != cudaSuccess) return e;
    FR_MARK(prof, "common_flux_g");
    mixed_common_flux(c->mx, c->dc.ph, true, uf, gf, s);
    for (int t = 0; t < np_; ++t)
      if (c->parts[t]->dc.nbnd) launch_common_flux_g(c->parts[t]->dc, uf + c->mx_fpo[t], gf + c->mx_fpo[t], false, s);
  } else {
    FR_MARK(prof, "common_flux");
    mixed_common_flux(c->mx, c->dc.ph, false, uf, nullptr, s);
    for (int t = 0; t < np_; ++t)
      if (c->parts[t]->dc.nbnd) launch_common_flux(c->parts[t]->dc, uf + c->mx_fpo[t], nullptr, false, s);
  }
  FR_MARK(prof, "el_fluxdiv");
  for (int t = 0; t < np_ && e == cudaSuccess; ++t)
    e = element_fluxdiv(c->parts[t]->dc, up(t), (const double *)(work + c->mx_qoff[t]), uf + c->mx_fpo[t], (char *)rhs + c->mx_soff[t], s);
  return e != cudaSuccess ? e : cudaGetLastError();
}

#define FR_NEED_READY(c, ret) \
  if (!(c)) return ret;      \
  if (!(c)->ready) { (c)->err = "fr_setup_operators has not completed"; return ret; }

#define FR_NOT_MIXED(c, what) \
  if (!(c)->parts.empty()) return fail(c, FR_EINVAL, what ": single-type query on a mixed-mesh context (use fr_part_info)");

int64_t fr_num_solution_points(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) FR_NOT_MIXED(c, "fr_num_solution_points") return c->ops.Nu; }
int64_t fr_num_flux_points(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) FR_NOT_MIXED(c, "fr_num_flux_points") return c->ops.Nf; }
int64_t fr_num_vars(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->dc.NV; }
int64_t fr_num_pairs(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->parts.empty() ? c->mc.npairs : c->mx.n; }
int64_t fr_leading_dim(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) FR_NOT_MIXED(c, "fr_leading_dim") return c->dc.ld; }
int64_t fr_state_bytes(const fr_ctx *c) {
  FR_NEED_READY(c, FR_EINVAL)
  if (!c->parts.empty()) return c->mx_state;
  return (int64_t)c->ops.Nu * c->dc.NV * c->dc.ld * (c->dc.f64 ? 8 : 4);
}
int64_t fr_num_parts(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->parts.empty() ? 1 : (int64_t)c->parts.size(); }
int fr_part_info(const fr_ctx *c, int part, fr_part_info_t *info) {
  FR_NEED_READY(c, FR_EINVAL)
  if (!info || part < 0 || part >= (c->parts.empty() ? 1 : (int)c->parts.size())) return fail(c, FR_EINVAL, "fr_part_info: part out of range or NULL output");
  const fr_ctx *q = c->parts.empty() ? c : c->parts[part];
  info->etype = q->ops.etype; info->reserved = 0;
  info->n_elems = q->mc.Nel; info->n_solution_points = q->ops.Nu; info->n_flux_points = q->ops.Nf; info->leading_dim = q->dc.ld;
  info->state_offset = c->parts.empty() ? 0 : c->mx_soff[part];
  return FR_OK;
}
int fr_part_solution_point_coords(const fr_ctx *c, int part, double *xyz) {
  FR_NEED_READY(c, FR_EINVAL)
  if (!xyz || part < 0 || part >= (c->parts.empty() ? 1 : (int)c->parts.size())) return fail(c, FR_EINVAL, "fr_part_solution_point_coords: part out of range or NULL buffer");
  const fr_ctx *q = c->parts.empty() ? c : c->parts[part];
  std::memcpy(xyz, q->mc.xu.data(), q->mc.xu.size() * sizeof(double));
  return FR_OK;
}
int64_t fr_workspace_bytes(const fr_ctx *c) { FR_NEED_READY(c, FR_EINVAL) return c->wl.total; }
int64_t fr_stepper_workspace_bytes(const fr_ctx *c, int stepper) {
  FR_NEED_READY(c, FR_EINVAL)
  const int regs = stepper == FR_STEPPER_EULER ? 1 : stepper == FR_STEPPER_RK4 ? 3 : stepper == FR_STEPPER_DOPRI5 ? 7 : -1;
  if (regs < 0) return fail(c, FR_EINVAL, "unknown stepper");
  return c->wl.reg0 + regs * c->wl.reg_stride;
}
int64_t fr_rhs_kernel_launches(const fr_ctx *c) {
  FR_NEED_READY(c, FR_EINVAL)
  if (!c->parts.empty()) {
    int64_t n = (int64_t)c->parts.size() * (c->dc.ns ? 3 : 2) + (c->mx.n ? (c->dc.ns ? 2 : 1) : 0);
    for (const fr_ctx *q : c->parts) if (q->dc.nbnd) n += c->dc.ns ? 2 : 1;
    return n;
  }
  return c->use_tensor ? tensor_rhs_launches(c->dc) : generic_rhs_launches(c->dc);
}

int fr_solution_point_coords(const fr_ctx *c, double *xyz) {
  FR_NEED_READY(c, FR_EINVAL)
  FR_NOT_MIXED(c, "fr_solution_point_coords")
  if (!xyz) return fail(c, FR_EINVAL, "xyz_host is NULL");
  std::memcpy(xyz, c->mc.xu.data(), c->mc.xu.size() * sizeof(double));
  return FR_OK;
}

int fr_operator_dims(const fr_ctx *c, int id, int64_t *rows, int64_t *cols) {
  FR_NEED_READY(c, FR_EINVAL)
  FR_NOT_MIXED(c, "fr_operator_dims")
  if (id < 0 || id > 6 || !rows || !cols) return fail(c, FR_EINVAL, "operator id out of range or NULL output");
  *rows = c->ops.rows[id]; *cols = c->ops.cols[id];
  return FR_OK;
}

int fr_get_operator(const fr_ctx *c, int id, double *buf) {
  FR_NEED_READY(c, FR_EINVAL)
  FR_NOT_MIXED(c, "fr_get_operator")
  if (id < 0 || id > 6 || !buf) return fail(c, FR_EINVAL, "operator id out of range or NULL buffer");
  std::memcpy(buf, c->ops.M[id].data(), c->ops.M[id].size() * sizeof(double));
  return FR_OK;
}

int fr_get_pairs(const fr_ctx *c, int32_t *pairs, double *normals, double *jn) {
  FR_NEED_READY(c, FR_EINVAL)
  FR_NOT_MIXED(c, "fr_get_pairs")
  if (c->lean) return fail(c, FR_EINVAL, "fr_get_pairs: host tables were released (FR_FLAG_LEAN)");
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
  FR_NOT_MIXED(c, "fr_get_metrics")
  if (c->lean) return fail(c, FR_EINVAL, "fr_get_metrics: host tables were released (FR_FLAG_LEAN)");
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
  if (!c->parts.empty()) {
    cudaError_t em = mixed_rhs(c, u, rhs, (char *)work, s, prof);
    if (em != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_rhs launch: ") + cudaGetErrorString(em));
    return FR_OK;
  }
  cudaError_t e = c->use_tensor ? tensor_rhs(c->dc, c->tp, u, rhs, (char *)work + c->wl.uf, s, prof)
                                : generic_rhs(c->dc, c->wl, u, rhs, (char *)work, s, prof);
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_rhs launch: ") + cudaGetErrorString(e));
  return FR_OK;
}

int fr_rhs(fr_ctx *c, const void *u, void *rhs, void *work, void *stream) { return rhs_impl(c, u, rhs, work, stream, nullptr); }

// ---- fr_rhs without a caller-owned workspace (include/fr.h): scratch in a static device array ----
// In host code `g_static_work` is a host-side stand-in of the device array, not a device address: the address is asked of the
// runtime once per device, with that device current, and cached.
static __device__ __align__(256) unsigned char g_static_work[FR_STATIC_WORK_BYTES];

static cudaError_t static_work_address(int dev, void **out) {
  static std::mutex mtx;
  static void *ptr[256] = {};
  if (dev < 0 || dev >= 256) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mtx);
  if (!ptr[dev]) {
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_work);  // the current device is `dev` (checked by the caller)
    if (e != cudaSuccess) return e;
    if (!p || ((uintptr_t)p & 255)) return cudaErrorInvalidSymbol;
    ptr[dev] = p;
  }
  *out = ptr[dev];
  return cudaSuccess;
}

int fr_rhs_static(fr_ctx *c, const void *u, void *rhs, void *stream) {
  FR_NEED_READY(c, FR_EINVAL)
  if (c->host_only) return fail(c, FR_EINVAL, "fr_rhs_static: context was set up with FR_FLAG_HOST_ONLY");
  if (c->wl.reg0 > (int64_t)FR_STATIC_WORK_BYTES)
    return fail(c, FR_ENOMEM, "fr_rhs_static: the right-hand side needs " + std::to_string(c->wl.reg0) + " bytes of scratch, the static array holds " +
                                  std::to_string((int64_t)FR_STATIC_WORK_BYTES) + " (FR_STATIC_WORK_BYTES): use fr_rhs with a caller-owned workspace");
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != c->dc.dev)
    return fail(c, FR_EINVAL, "fr_rhs_static: the current CUDA device is not the one fr_setup_operators uploaded the constants to");
  void *work = nullptr;
  cudaError_t e = static_work_address(dev, &work);
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_rhs_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
  return rhs_impl(c, u, rhs, work, stream, nullptr);
}

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

// ---- time steppers (Table 1 :263).  Registers: work + reg0 + i * reg_stride ----
// out1 = sum a_i in_i, out2 = sum b_i in_i over the state matrices of the context (every part of a mixed mesh)
static cudaError_t ctx_lincomb(const fr_ctx *c, int nin, const void *const *in, const double *a, const double *b, void *out1, void *out2,
                               cudaStream_t s) {
  const bool f64 = c->dc.f64;
  if (c->parts.empty()) return rk_lincomb(f64, (int64_t)c->ops.Nu * c->dc.NV, c->dc.ld, c->dc.Nel, nin, in, a, b, out1, out2, s);
  cudaError_t e = cudaSuccess;
  for (size_t t = 0; t < c->parts.size() && e == cudaSuccess; ++t) {
    const fr_ctx *q = c->parts[t];
    const void *inp[RK_MAX_IN];
    for (int i = 0; i < nin; ++i) inp[i] = (const char *)in[i] + c->mx_soff[t];
    e = rk_lincomb(f64, (int64_t)q->ops.Nu * q->dc.NV, q->dc.ld, q->dc.Nel, nin, inp, a, b, out1 ? (char *)out1 + c->mx_soff[t] : nullptr,
                   out2 ? (char *)out2 + c->mx_soff[t] : nullptr, s);
  }
  return e;
}

#define FR_STEPPER_PROLOGUE(name)                                                                       \
  FR_NEED_READY(c, FR_EINVAL)                                                                           \
  if (c->host_only) return fail(c, FR_EINVAL, name ": context was set up with FR_FLAG_HOST_ONLY");       \
  if (!u || !work) return fail(c, FR_EINVAL, name ": NULL device pointer");                              \
  cudaStream_t s = (cudaStream_t)stream;                                                                \
  char *wk = (char *)work;                                                                              \
  auto reg = [&](int i) { return (void *)(wk + c->wl.reg0 + i * c->wl.reg_stride); };                   \
  int rc;                                                                                               \
  cudaError_t e = cudaSuccess;

int fr_rk4_step(fr_ctx *c, void *u, double dt, void *work, void *stream) {
  FR_STEPPER_PROLOGUE("fr_rk4_step")
  void *k = reg(0), *tmp = reg(1), *acc = reg(2);
  const void *in[3] = {u, k, acc};
  // k1; tmp = u + dt/2 k1; acc = u + dt/6 k1
  if ((rc = fr_rhs(c, u, k, work, stream)) != FR_OK) return rc;
  { const double a[2] = {1, dt / 2}, b[2] = {1, dt / 6}; e = ctx_lincomb(c, 2, in, a, b, tmp, acc, s); }
  // k2; tmp = u + dt/2 k2; acc += dt/3 k2
  if (e == cudaSuccess && (rc = fr_rhs(c, tmp, k, work, stream)) != FR_OK) return rc;
  if (e == cudaSuccess) { const double a[3] = {1, dt / 2, 0}, b[3] = {0, dt / 3, 1}; e = ctx_lincomb(c, 3, in, a, b, tmp, acc, s); }
  // k3; tmp = u + dt k3; acc += dt/3 k3
  if (e == cudaSuccess && (rc = fr_rhs(c, tmp, k, work, stream)) != FR_OK) return rc;
  if (e == cudaSuccess) { const double a[3] = {1, dt, 0}, b[3] = {0, dt / 3, 1}; e = ctx_lincomb(c, 3, in, a, b, tmp, acc, s); }
  // k4; u = acc + dt/6 k4
  if (e == cudaSuccess && (rc = fr_rhs(c, tmp, k, work, stream)) != FR_OK) return rc;
  if (e == cudaSuccess) { const double a[3] = {0, dt / 6, 1}; e = ctx_lincomb(c, 3, in, a, nullptr, u, nullptr, s); }
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_rk4_step launch: ") + cudaGetErrorString(e));
  return FR_OK;
}

int fr_euler_step(fr_ctx *c, void *u, double dt, void *work, void *stream) {
  FR_STEPPER_PROLOGUE("fr_euler_step")
  void *k = reg(0);
  if ((rc = fr_rhs(c, u, k, work, stream)) != FR_OK) return rc;
  const void *in[2] = {u, k};
  const double a[2] = {1.0, dt};
  e = ctx_lincomb(c, 2, in, a, nullptr, u, nullptr, s);
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_euler_step launch: ") + cudaGetErrorString(e));
  return FR_OK;
}

int fr_dopri5_step(fr_ctx *c, void *u, double dt, void *work, void *stream, double *err_dev) {
  FR_STEPPER_PROLOGUE("fr_dopri5_step")
  if (err_dev && !c->parts.empty()) return fail(c, FR_EUNSUPPORTED, "fr_dopri5_step: the error norm is not available on mixed meshes (pass NULL)");
  // Dormand-Prince 5(4), reading A24.  Row i+1 of A gives the state of stage i+1; row 7 = the fifth-order weights (FSAL).
  static const double A[7][6] = {
      {0, 0, 0, 0, 0, 0},
      {1.0 / 5, 0, 0, 0, 0, 0},
      {3.0 / 40, 9.0 / 40, 0, 0, 0, 0},
      {44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0},
      {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0},
      {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0},
      {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}};
  static const double B4[7] = {5179.0 / 57600, 0, 7571.0 / 16695, 393.0 / 640, -92097.0 / 339200, 187.0 / 2100, 1.0 / 40};
  void *tmp = reg(6);  // registers 0..5 hold k1..k6; k7 = R(u_new) overwrites k2, whose weights are zero in both rules
  if ((rc = fr_rhs(c, u, reg(0), work, stream)) != FR_OK) return rc;
  for (int i = 1; i < 6 && e == cudaSuccess; ++i) {
    const void *in[7] = {u, reg(0), reg(1), reg(2), reg(3), reg(4), reg(5)};
    double a[7] = {1.0, 0, 0, 0, 0, 0, 0};
    for (int j = 0; j < i; ++j) a[1 + j] = dt * A[i][j];
    e = ctx_lincomb(c, 1 + i, in, a, nullptr, tmp, nullptr, s);
    if (e == cudaSuccess && (rc = fr_rhs(c, tmp, reg(i), work, stream)) != FR_OK) return rc;
  }
  if (e == cudaSuccess) {  // u <- u + dt sum b5_i k_i ; tmp <- dt sum (b5_i - b4_i) k_i without k7
    const void *in[7] = {u, reg(0), reg(1), reg(2), reg(3), reg(4), reg(5)};
    double a[7] = {1.0, 0, 0, 0, 0, 0, 0}, b[7] = {0, 0, 0, 0, 0, 0, 0};
    for (int j = 0; j < 6; ++j) { a[1 + j] = dt * A[6][j]; b[1 + j] = dt * (A[6][j] - B4[j]); }
    e = ctx_lincomb(c, 7, in, a, err_dev ? b : nullptr, u, err_dev ? tmp : nullptr, s);
  }
  if (err_dev && e == cudaSuccess) {
    if ((rc = fr_rhs(c, u, reg(1), work, stream)) != FR_OK) return rc;  // k7
    const void *in[2] = {tmp, reg(1)};
    const double a[2] = {1.0, -dt * B4[6]};  // + dt (b5_7 - b4_7) k7, b5_7 = 0
    e = ctx_lincomb(c, 2, in, a, nullptr, tmp, nullptr, s);
    // RMS of the error estimate = distance of tmp from a zero register (k7's, no longer needed)
    if (e == cudaSuccess) { const void *z[1] = {tmp}; const double za[1] = {0.0}; e = ctx_lincomb(c, 1, z, za, nullptr, reg(1), nullptr, s); }
    if (e == cudaSuccess)
      e = rk_rms_diff(c->dc.f64, (int64_t)c->ops.Nu * c->dc.NV, c->dc.ld, c->dc.Nel, tmp, reg(1), (double *)(wk + c->wl.partials), err_dev, s);
  }
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_dopri5_step launch: ") + cudaGetErrorString(e));
  return FR_OK;
}

int fr_state_lincomb(fr_ctx *c, int n_in, const void *const *in, const double *coef, void *out, void *stream) {
  FR_NEED_READY(c, FR_EINVAL)
  if (c->host_only) return fail(c, FR_EINVAL, "fr_state_lincomb: context was set up with FR_FLAG_HOST_ONLY");
  if (n_in < 1 || n_in > RK_MAX_IN || !in || !coef || !out) return fail(c, FR_EINVAL, "fr_state_lincomb: bad arguments");
  for (int i = 0; i < n_in; ++i) if (!in[i]) return fail(c, FR_EINVAL, "fr_state_lincomb: NULL operand");
  cudaError_t e = ctx_lincomb(c, n_in, in, coef, nullptr, out, nullptr, (cudaStream_t)stream);
  if (e != cudaSuccess) return fail(c, FR_ECUDA, std::string("fr_state_lincomb launch: ") + cudaGetErrorString(e));
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
  for (fr_ctx *q : c->parts) free_dev(q);
  free_dev(c);
  delete c;
}

const char *fr_last_error(const fr_ctx *c) { return c ? c->err.c_str() : g_setup_err.c_str(); }

}  // extern "C"
