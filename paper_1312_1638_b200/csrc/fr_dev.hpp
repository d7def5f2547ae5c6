// Device-side constant tables of a context and the launch entry points of the two kernel families.
#pragma once
#include <cuda_runtime.h>

#include <cstdint>

#include "fr_physics.cuh"

namespace fr {

// one bit per device ordinal (cudaFuncSetAttribute is per device)
struct DevFlags {
  uint64_t bits[4] = {0, 0, 0, 0};
  bool test(int d) const { return d >= 0 && d < 256 && ((bits[d >> 6] >> (d & 63)) & 1u); }
  void set(int d) { if (d >= 0 && d < 256) bits[d >> 6] |= 1ull << (d & 63); }
};

struct DevConsts {
  int nd, NV, Nu, Nf, n, nfp, etype;
  int dev;       // device ordinal the constants were uploaded to (fr_setup_operators); fr_rhs refuses any other current device
  int64_t Nel, ld, npairs, nbnd;
  bool ns;       // Navier-Stokes (gradients, LDG) or Euler
  bool f64;      // storage precision of u / rhs
  bool staged;   // FR_FLAG_FORCE_GENERIC: the paper's staged kernel sequence, no fused kernels
  bool force_el; // part of a mixed mesh: always the fused element kernels (quadrilaterals p = 4 too)
  bool affine;   // every element has constant metric terms (straight-sided simplices, parallelepipeds): one point serves all
  bool aff;      // blk and every element affine: smat / rcpj hold ONE point per element ([block][9][FR_BLK], [block][1][FR_BLK])
  bool blk;      // library-internal arrays are element-blocked (FR_BLK elements per block), see fp_row()
  Phys ph;
  // dense operators (device, row-major doubles)
  const double *M0, *M3, *M6, *M46, *M132;
  const double *hM0, *hM3, *hM6, *hM46, *hM132;  // host copies (owned by the context): operators passed as kernel parameters
  // metrics at solution points
  const double *smat;   // [nd*nd][Nu][ld]
  const double *rcpj;   // [Nu][ld]
  // flux-point pairs in iteration order
  const int32_t *pLs, *pLe, *pRs, *pRe;
  const double *pn, *pJnL, *pJnR;
  // boundary flux points
  const int32_t *bs, *be, *bbc;
  const double *bn, *bJn;
  const BcDev *bcs;
  int nbcs;
  // element-centric tables (tensor-product kernels)
  const int32_t *fp_pe, *fp_ps;
  void *map_cache;           // host object owned by the context (fr_tma.cuh: MapCache): encoded tensor maps keyed on the caller's pointers
  const int64_t *fp_poff;    // hexahedral TMA path, [block][Nf][FR_BLK]: offset of the partner's first variable in U^f, or -1 - bc_id
  const uint8_t *face_code;  // [6][ld] (hexahedra): 0 = face without LDG weight, 1 = L side, 2 = R side, 3 = boundary (fr_hex_tma.cu)
  const double *fp_n, *fp_Jn;
  // affine hexahedral meshes on the TMA path (aff): the unit normal and J n of a flux point are those of its face, so the pair
  // kernels read them from per-face tables [nd][2 nd][ld] / [2 nd][ld] (storage precision; re-read from cache by the N^2 flux
  // points of a face) instead of the per-pair tables pn / pJnL / pJnR.  NULL: per-pair tables.
  const double *pf_n, *pf_Jn;
};

// Element-blocked layout of library-internal arrays (flux-point arrays U^f / D~, jumps, G^f, Q, and the metric / normal
// tables of the hexahedral TMA path).  The caller-visible layout [row][ld] puts consecutive rows ld*8 bytes apart: at
// 10^6 elements every row of a CTA's working set lies in a page of its own and the TMA kernels run at less than half
// speed (measured).  Internal arrays therefore use [element block][row][FR_BLK]: all rows that belong
// to FR_BLK consecutive elements are contiguous.  u and rhs keep the ABI layout.
constexpr int FR_BLK = 32;

// start of row `row` (of `rows` per element) for element e, and the distance between consecutive rows of one element
__host__ __device__ inline size_t fp_row(bool blk, int64_t ld, int rows, int row, int64_t e) {
  return blk ? ((size_t)(e / FR_BLK) * rows + row) * FR_BLK + (size_t)(e % FR_BLK) : (size_t)row * ld + e;
}
__host__ __device__ inline size_t fp_rstride(bool blk, int64_t ld) { return blk ? (size_t)FR_BLK : (size_t)ld; }

// Workspace layout (doubles unless noted); offsets in bytes from work_dev
struct WorkLayout {
  int64_t uf, cf, qu, qf;          // generic path: U^f (-> D~), C^f, Q~ -> Q -> F~, Q^f
  int64_t partials;                // RK_MAX_PARTIALS doubles (error norm of fr_dopri5_step)
  int64_t reg0, reg_stride;        // stepper registers in the storage precision: reg0 + i * reg_stride, i < 7
  int64_t total;                   // through register 2 (fr_rk4_step)
};

// Optional per-kernel timing: an event is recorded before every kernel and after the last one.
struct Prof {
  static const int MAXK = 32;
  cudaEvent_t ev[MAXK + 1];
  const char *names[MAXK];
  int n = 0;
  cudaStream_t s = nullptr;
  void mark(const char *name) { if (n < MAXK) { names[n] = name; cudaEventRecord(ev[n], s); ++n; } }
  void end() { cudaEventRecord(ev[n], s); }
};
#define FR_MARK(prof, name) do { if (prof) (prof)->mark(name); } while (0)

// generic (staged, dense-operator) path: any element type.  Returns cudaGetLastError().
cudaError_t generic_rhs(const DevConsts &c, const WorkLayout &w, const void *u, void *rhs, char *work, cudaStream_t s, Prof *prof);
int generic_rhs_launches(const DevConsts &c);
// point-wise / pair kernels of the generic path reused by the tensor-product path
void launch_common_jump(const DevConsts &c, const double *uf, double *cf, cudaStream_t s);  // {C - u^f} of Eq 9
void launch_common_sol(const DevConsts &c, const double *uf, double *cf, cudaStream_t s);   // C of Eq 7 (2-D element kernels)
void launch_tflux(const DevConsts &c, const void *u, double *qu, cudaStream_t s);           // Eq 12, in place over Q^u
void launch_common_flux(const DevConsts &c, void *uf, const void *qf, bool f32, cudaStream_t s);  // Eq 15-17, in place over U^f (f32: float arrays)

// register updates of the time steppers (fr_rk.cu): rows x ld matrices of which the first nel columns are updated
constexpr int RK_MAX_IN = 8;
constexpr int RK_MAX_PARTIALS = 4096;
// out1 = sum_i a[i] in[i], out2 = sum_i b[i] in[i]  (either output may be NULL or alias an input)
cudaError_t rk_lincomb(bool f64, int64_t rows, int64_t ld, int64_t nel, int nin, const void *const *in, const double *a, const double *b,
                       void *out1, void *out2, cudaStream_t s);
// *out = sqrt(mean (x - y)^2) over the rows x nel values, deterministic; part: RK_MAX_PARTIALS doubles of scratch
cudaError_t rk_rms_diff(bool f64, int64_t rows, int64_t ld, int64_t nel, const void *x, const void *y, double *part, double *out,
                        cudaStream_t s);

}  // namespace fr
