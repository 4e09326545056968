// tdde_create.cu -- tdde_create / tdde_destroy: validation, band repacking, per-class banded LU (host, one-time),
// device allocation.  SURVEY 8(a) a0; PAPER.md:211-215 (Eq. 26), :268, :275-276 ("performed at start-up").
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include "tdde_handle.h"
#include "tdde_partition.h"

thread_local std::string g_last_cuda_error;

int tdde_cuda_fail(cudaError_t e, const char* what) {
  g_last_cuda_error = std::string(cudaGetErrorName(e)) + ": " + cudaGetErrorString(e) + " in " + what;
  cudaGetLastError();
  return e == cudaErrorMemoryAllocation ? TDDE_ENOMEM : TDDE_ECUDA;
}

namespace {

template <class T>
int dev_upload(T** dst, const T* src, size_t count, cudaStream_t s) {
  *dst = nullptr;
  if (count == 0) count = 1, src = nullptr;
  CU(cudaMalloc((void**)dst, count * sizeof(T)));
  if (src) CU(cudaMemcpyAsync(*dst, src, count * sizeof(T), cudaMemcpyHostToDevice, s));
  else CU(cudaMemsetAsync(*dst, 0, count * sizeof(T), s));
  return 0;
}

// row-band [n][2w+1] (band[i][d+w] = M[i][i+d]) -> column-band col[j][e] = M[j-w+e][j], zero outside the matrix
void row_to_col_band(const zc* row, zc* col, int n, int w) {
  const int nd = 2 * w + 1;
  for (int j = 0; j < n; ++j)
    for (int e = 0; e < nd; ++e) {
      const int i = j - w + e;
      col[(size_t)j * nd + e] = (i >= 0 && i < n) ? row[(size_t)i * nd + (2 * w - e)] : zc(0, 0);
    }
}

// same, into a wider column band of half-width W >= w (entries beyond w are zero)
void row_to_col_band_padded(const zc* row, zc* col, int n, int w, int W) {
  const int nd = 2 * w + 1, ND = 2 * W + 1;
  for (int j = 0; j < n; ++j)
    for (int e = 0; e < ND; ++e) {
      const int i = j - W + e;
      col[(size_t)j * ND + e] = (i >= 0 && i < n && std::abs(i - j) <= w) ? row[(size_t)i * nd + (j - i + w)] : zc(0, 0);
    }
}

int validate(const tdde_config* c, const tdde_c64* S, const tdde_c64* H0, const int32_t* cls, const tdde_term* terms) {
  if (!c || !S || !H0 || !cls) return TDDE_EINVAL;
  if (c->n_ang <= 0 || c->n_rad <= 0 || c->n_cls <= 0 || c->n_cls > c->n_ang) return TDDE_EINVAL;
  if (c->w0 < 1 || c->w0 > 32 || c->w0 >= c->n_rad) return TDDE_EINVAL;
  if (c->n_terms < 0 || c->n_terms > TDDE_MAX_TERMS || (c->n_terms > 0 && !terms)) return TDDE_EINVAL;
  if (c->max_iter <= 0 || !(c->rtol >= 0) || !std::isfinite(c->dt) || c->dt == 0.0) return TDDE_EINVAL;
  if ((long long)c->n_ang * c->n_rad > (1LL << 40)) return TDDE_EINVAL;
  for (int a = 0; a < c->n_ang; ++a)
    if (cls[a] < 0 || cls[a] >= c->n_cls) return TDDE_EINVAL;
  for (int L = 0; L < c->n_terms; ++L) {
    const tdde_term& t = terms[L];
    if (t.w < 0 || t.w > 32 || t.w >= c->n_rad || !t.R_band || !t.A_rowptr) return TDDE_EINVAL;
    if (t.A_rowptr[0] != 0) return TDDE_EINVAL;
    for (int a = 0; a < c->n_ang; ++a)
      if (t.A_rowptr[a + 1] < t.A_rowptr[a]) return TDDE_EINVAL;
    const int nnz = t.A_rowptr[c->n_ang];
    if (nnz > 0 && (!t.A_col || !t.A_val)) return TDDE_EINVAL;
    for (int q = 0; q < nnz; ++q)
      if (t.A_col[q] < 0 || t.A_col[q] >= c->n_ang) return TDDE_EINVAL;
  }
  return 0;
}

// Structure fit for the register-resident banded kernel: every A_L non-zero only at channel offsets 1 <= |o| <= m_L (no diagonal,
// no duplicates).  The kernels are instantiated for a few shapes (T, m_L = M0 + MS L, W); the problem fits a shape when it has no more
// terms, each term's reach is covered by a distinct slot, and every band is no wider than W.  The cheapest fitting shape is taken;
// unused slots, unused offsets and the extra diagonals are zero-filled (wasted FMAs, but no change of kernel).
struct BandFit { int T, m0, ms, W, slot_of[TDDE_MAX_TERMS]; };

bool fit_banded(const tdde_config* c, const tdde_term* terms, BandFit* f) {
  const int T = c->n_terms;
  int reach[TDDE_MAX_TERMS], order[TDDE_MAX_TERMS], maxw = c->w0;
  for (int L = 0; L < T; ++L) {
    maxw = std::max(maxw, (int)terms[L].w);
    reach[L] = 0;
    for (int a = 0; a < c->n_ang; ++a)
      for (int q = terms[L].A_rowptr[a]; q < terms[L].A_rowptr[a + 1]; ++q) {
        const int o = terms[L].A_col[q] - a;
        if (o == 0) return false;
        reach[L] = std::max(reach[L], std::abs(o));
        for (int q2 = terms[L].A_rowptr[a]; q2 < q; ++q2)       // duplicates would need summing (the staged path does)
          if (terms[L].A_col[q] == terms[L].A_col[q2]) return false;
      }
    order[L] = L;
  }
  std::sort(order, order + T, [&](int x, int y) { return reach[x] < reach[y] || (reach[x] == reach[y] && x < y); });
  int shapes[64][4];
  const int ns = apply_banded_shapes(shapes, 64);
  long long best = -1;
  for (int s = 0; s < ns; ++s) {
    const int Tt = shapes[s][0], m0 = shapes[s][1], ms = shapes[s][2], W = shapes[s][3];
    if (W < maxw || Tt < T || (T > 0 && Tt == 0) || (T == 0 && Tt != 0)) continue;
    if (!apply_banded_available(0, 0, 0, W)) continue;           // the S-only apply needs the T = 0 kernel of the same width
    int slot_of[TDDE_MAX_TERMS], next = 0;
    bool ok = true;
    for (int i = 0; i < T && ok; ++i) {                          // slots and terms both ascending in reach: greedy is optimal
      while (next < Tt && m0 + ms * next < reach[order[i]]) ++next;
      if (next >= Tt) ok = false; else slot_of[order[i]] = next++;
    }
    if (!ok) continue;
    long long cost = 2 * W + 1;
    for (int L = 0; L < Tt; ++L) cost += 2 * W + 1 + 2 * (m0 + ms * L);
    if (best < 0 || cost < best) {
      best = cost;
      f->T = Tt; f->m0 = m0; f->ms = ms; f->W = W;
      for (int L = 0; L < T; ++L) f->slot_of[L] = slot_of[L];
    }
  }
  return best >= 0;
}

}  // namespace

extern "C" void tdde_destroy(tdde_handle* h) {
  if (!h) return;
  DeviceGuard dg(h->device);
  cudaStreamSynchronize(h->stream);
  void* ptrs[] = {h->d_cls, h->d_S, h->d_H0, h->d_Mp, h->d_blk_tmp, h->d_Aoff, h->d_Rall, h->d_Rfrag, h->d_slot, h->d_cta_cls, h->d_eig, h->d_proj, h->d_pslot, h->d_warp_cls, h->d_spval, h->d_spcol, h->d_Wsp, h->d_Corner, h->d_Schur, h->d_rsm, h->d_rsp, h->d_Lcol, h->d_Ucol, h->X, h->r,
                  h->rhat, h->p, h->v, h->s, h->t, h->y, h->z, h->c_stage, h->d_st, h->d_st_bench, h->d_partials,
                  h->d_ticket, h->d_g, h->d_g_small, h->d_zero_g};
  for (void* p : ptrs) if (p) cudaFree(p);
  for (int L = 0; L < TDDE_MAX_TERMS; ++L) {
    if (h->d_R[L]) cudaFree(h->d_R[L]);
    if (h->d_Arowptr[L]) cudaFree(h->d_Arowptr[L]);
    if (h->d_Acol[L]) cudaFree(h->d_Acol[L]);
    if (h->d_Aval[L]) cudaFree(h->d_Aval[L]);
  }
  if (h->step_exec) cudaGraphExecDestroy(h->step_exec);
  if (h->cap) cudaStreamDestroy(h->cap);
  if (h->h_st) cudaFreeHost(h->h_st);
  cudaGetLastError();
  delete h;
}

static int create_impl(tdde_handle* h, const tdde_c64* S_band, const tdde_c64* H0_band, const int32_t* cls_of_chan,
                       const tdde_term* terms) {
  cudaStream_t s = h->stream;
  // ---- which apply kernel (by the structure of the A_L) ----
  h->user_terms = h->cfg.n_terms;
  for (int L = 0; L < TDDE_MAX_TERMS; ++L) h->term_slot[L] = L;
  BandFit fit;
  h->path = fit_banded(&h->cfg, terms, &fit) ? 1 : 0;
  if (const char* env = std::getenv("TDDE_APPLY_PATH")) { if (std::atoi(env) != 1) h->path = 0; }   // tests: force a lower tier
  // banded path: re-slot the terms into the fitted shape; empty slots become zero terms (R = 0, A empty, g = 0)
  std::vector<tdde_term> slotted;
  std::vector<zc> zero_band((size_t)h->cfg.n_rad * 3, zc(0, 0));
  std::vector<int32_t> zero_rowptr((size_t)h->cfg.n_ang + 1, 0);
  if (h->path == 1) {
    slotted.assign(std::max(fit.T, 1), tdde_term{1, 0, reinterpret_cast<const tdde_c64*>(zero_band.data()), zero_rowptr.data(), nullptr, nullptr});
    for (int L = 0; L < h->user_terms; ++L) { slotted[fit.slot_of[L]] = terms[L]; h->term_slot[L] = fit.slot_of[L]; }
    h->g_identity = fit.T == h->user_terms;
    for (int L = 0; L < h->user_terms; ++L) h->g_identity = h->g_identity && fit.slot_of[L] == L;
    h->cfg.n_terms = fit.T;
    terms = slotted.data();
  }
  const tdde_config& c = h->cfg;
  const int n_rad = c.n_rad, w0 = c.w0, nd0 = 2 * w0 + 1, T = c.n_terms;
  h->ld = (c.n_ang + 31) / 32 * 32;
  h->nint = (long long)n_rad * h->ld;
  h->n = (long long)c.n_ang * n_rad;
  h->tau = 0.5 * c.dt;

  CU(cudaGetDevice(&h->device));
  CU(cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, h->device));
  const int m0 = h->path == 1 ? fit.m0 : 0, ms = h->path == 1 ? fit.ms : 0;
  h->bT = T; h->bM0 = m0; h->bMS = ms; h->bW = h->path == 1 ? fit.W : w0;
  // Term split over two warp groups (256-thread CTA, one per SM, 255 registers each): measured on B200 it wins once
  // the per-thread A_L registers no longer fit (HBM-scale, T = 7: 3.21 -> 2.39 ms) and loses below (Large, T = 5:
  // 0.31 -> 0.37 ms), so it is chosen by the number of terms.
  h->apply_ng = (T >= 6) ? 2 : 1;
  if (const char* env = std::getenv("TDDE_APPLY_NG")) h->apply_ng = std::atoi(env) == 2 ? 2 : 1;

  // Staged sparse-A path (tdde_apply_sparse.cu) for everything the register-A kernel does not cover: general sparse A_L
  // (ELL rows in shared memory), any T, per-term bandwidths padded to one of the instantiated widths.
  std::vector<zc> ell_val;
  std::vector<int> ell_col;
  if (h->path == 0) {
    int maxw = w0;
    for (int L = 0; L < T; ++L) maxw = std::max(maxw, (int)terms[L].w);
    const int widths[4] = {3, 6, 9, 13};
    int spW = 0;
    for (int q = 0; q < 4 && !spW; ++q) if (maxw <= widths[q]) spW = widths[q];
    if (spW) {
      // ELL rows (duplicate columns of a CSR row summed), the coupling reach, the tile width
      int nslots = 0, reach = 0;
      std::vector<std::vector<std::pair<int, zc>>> rows((size_t)T * c.n_ang);
      for (int L = 0; L < T; ++L) {
        const zc* val = reinterpret_cast<const zc*>(terms[L].A_val);
        int mx = 0;
        for (int a = 0; a < c.n_ang; ++a) {
          auto& row = rows[(size_t)L * c.n_ang + a];
          for (int q = terms[L].A_rowptr[a]; q < terms[L].A_rowptr[a + 1]; ++q) {
            const int col = terms[L].A_col[q];
            size_t k = 0;
            while (k < row.size() && row[k].first != col) ++k;
            if (k == row.size()) row.push_back({col, val[q]}); else row[k].second += val[q];
            reach = std::max(reach, std::abs(col - a));
          }
          mx = std::max(mx, (int)row.size());
        }
        h->sp_nslot[L] = mx;
        nslots += mx;
      }
      const bool full = TDDE_AP_NC + 2 * reach >= h->ld;
      const int xw = full ? h->ld : TDDE_AP_NC + 2 * reach;
      const size_t cap = (size_t)220 * 1024;
      const bool a_smem = apply_sparse_smem(spW, T, nslots, xw, true) <= cap && !std::getenv("TDDE_SPARSE_A_GLOBAL");
      if ((a_smem || apply_sparse_smem(spW, T, nslots, xw, false) <= cap) && !std::getenv("TDDE_NO_STAGED")) {
        h->path = 2; h->spW = spW; h->sp_a_smem = a_smem ? 1 : 0; h->sp_nslots = nslots; h->sp_xw = xw; h->sp_full = full ? 1 : 0; h->sp_reach = reach;
        ell_val.assign((size_t)std::max(nslots, 1) * h->ld, zc(0, 0));
        ell_col.assign((size_t)std::max(nslots, 1) * h->ld, 0);
        int base = 0;
        for (int L = 0; L < T; ++L) {
          for (int a = 0; a < h->ld; ++a)
            for (int q = 0; q < h->sp_nslot[L]; ++q) {
              const bool have = a < c.n_ang && q < (int)rows[(size_t)L * c.n_ang + a].size();
              ell_val[(size_t)(base + q) * h->ld + a] = have ? rows[(size_t)L * c.n_ang + a][q].second : zc(0, 0);
              ell_col[(size_t)(base + q) * h->ld + a] = have ? rows[(size_t)L * c.n_ang + a][q].first : a;
            }
          base += h->sp_nslot[L];
        }
      }
    }
  }
  h->norm_banded = (h->path != 0);
  const int wpad = h->path == 2 ? h->spW : h->bW;          // half-width of the column bands the apply kernels read
  const int ndp = 2 * wpad + 1;
  h->blk_count = (long long)c.n_cls * n_rad * ndp;

  // radial segment length (structured paths): every segment recomputes 2 W halo rows.  Pick the segment count that
  // minimises waves x (rows + halo) over the resident CTA slots.
  {
    const int chan_blocks = (h->ld + TDDE_AP_NC - 1) / TDDE_AP_NC;
    const int per_sm = h->path == 2 ? 1 : (h->apply_ng == 2 ? TDDE_AP_MINB2 : TDDE_AP_MINB);
    const int slots = h->num_sms * per_sm;
    long long best_cost = -1;
    int best_seg = n_rad;
    // a segment may be shorter than its 2 W halo rows: on a problem that cannot fill the SMs otherwise, recomputing halo rows on idle
    // SMs is cheaper than leaving them idle (the cost below still counts the halo, so large problems keep long segments)
    int min_seg = 4;
    if (const char* env = std::getenv("TDDE_MIN_SEG")) min_seg = std::max(1, std::atoi(env));
    for (int segs = 1; segs <= n_rad; ++segs) {
      const int seg = (n_rad + segs - 1) / segs;
      if (seg < min_seg && segs > 1) break;
      const int real_segs = (n_rad + seg - 1) / seg;
      const long long ctas = (long long)chan_blocks * real_segs;
      const long long waves = (ctas + slots - 1) / slots;
      const long long cost = waves * (seg + 2 * wpad);
      if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_seg = seg; }
    }
    h->seg_len = best_seg;
    // the S-only apply has 13 complex FMAs per element: not ALU-bound, so halo recomputation is cheap and
    // many short segments (about 4 waves of 3 CTAs per SM) hide the TMA latency instead
    const int want = (4 * h->num_sms * 3 + chan_blocks - 1) / chan_blocks;
    h->seg_len_s = h->path == 2 ? h->seg_len : std::min(n_rad, std::max(4 * w0, (n_rad + want - 1) / want));
  }

  const zc* S = reinterpret_cast<const zc*>(S_band);
  const zc* H0 = reinterpret_cast<const zc*>(H0_band);
  const size_t blk_sz = (size_t)n_rad * nd0;

  // classes per channel (pads -> class 0)
  {
    std::vector<int> cls(h->ld, 0);
    for (int a = 0; a < c.n_ang; ++a) cls[a] = cls_of_chan[a];
    int rc = dev_upload(&h->d_cls, cls.data(), cls.size(), s);
    if (rc) return rc;
    CU(cudaStreamSynchronize(s));
  }
  // preconditioner: per warp (32 consecutive channels) the first TDDE_PC_MAXC distinct classes are staged
  {
    const int n_warp = h->ld / 32;
    std::vector<int> slot(h->ld, -1), wcls((size_t)n_warp * TDDE_PC_MAXC, -1);
    for (int b = 0; b < n_warp; ++b) {
      int cnt = 0;
      for (int a = b * 32; a < (b + 1) * 32; ++a) {
        const int k = a < c.n_ang ? cls_of_chan[a] : 0;
        int q = 0;
        while (q < cnt && wcls[(size_t)b * TDDE_PC_MAXC + q] != k) ++q;
        if (q == cnt && cnt < TDDE_PC_MAXC) wcls[(size_t)b * TDDE_PC_MAXC + cnt++] = k;
        slot[a] = q < cnt ? q : -1;
      }
    }
    int rc;
    if ((rc = dev_upload(&h->d_pslot, slot.data(), slot.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_warp_cls, wcls.data(), wcls.size(), s))) return rc;
    CU(cudaStreamSynchronize(s));
  }
  // block bands S, H0, M+ in the layout of the chosen path; LU of M+
  {
    const size_t blk_p = (size_t)n_rad * ndp;                // per-class size in the apply kernels' layout
    std::vector<zc> Sx(h->blk_count), Hx(h->blk_count), Mx(h->blk_count);
    std::vector<zc> Lc((size_t)c.n_cls * n_rad * w0), Uc((size_t)c.n_cls * n_rad * (w0 + 1));
    // preconditioner partitions: interiors short enough that a (32 channels x interior) tile plus the factor ring fits
    // several times into an SM's shared memory (k_precond_tile keeps the right-hand side on chip between its sweeps)
    const bool templated_w = w0 <= TDDE_PC_MAXW;
    int rows = w0 <= 4 ? 40 : w0 <= 9 ? 48 : 64;
    // small problems (the ones below the fused update kernels' threshold) cannot fill the SMs with (32 channels x interior) tiles of that
    // length: shorter interiors, i.e. more of them (measured: Medium 0.397 -> 0.373 ms per step, hydrogen 0.438 -> 0.42, Tiny 0.219 -> 0.21)
    if (h->nint < (1LL << 21)) rows = w0 <= 9 ? 24 : 28;
    if (const char* env = std::getenv("TDDE_PC_ROWS")) rows = std::max(1, std::atoi(env));
    int P = templated_w ? partitions_for_rows(n_rad, w0, rows) : 1;
    if (const char* env = std::getenv("TDDE_PC_PARTS")) P = templated_w ? std::max(1, std::atoi(env)) : 1;
    PartitionPlan plan = make_partition_plan(n_rad, w0, P);
    // a single interior must still fit the tile: force a split when it does not (always possible for n_rad that large)
    while (templated_w && precond_tile_smem(w0, plan.max_interior()) > (size_t)200 * 1024) {
      const PartitionPlan finer = make_partition_plan(n_rad, w0, plan.P + 1);
      if (finer.P == plan.P) return TDDE_EINVAL;
      plan = finer;
    }
    h->pc_P = plan.P; h->pc_tile_rows = plan.max_interior();
    h->pc_base = (n_rad - (plan.P - 1) * w0) / plan.P; h->pc_rem = (n_rad - (plan.P - 1) * w0) % plan.P;
    const size_t ww = (size_t)w0 * w0;
    const int nsep = plan.P - 1;
    std::vector<zc> Wsp(plan.P > 1 ? (size_t)c.n_cls * n_rad * 2 * w0 : 1), Corner(plan.P > 1 ? (size_t)c.n_cls * plan.P * 2 * ww : 1),
        Schur(plan.P > 1 ? (size_t)c.n_cls * nsep * 3 * ww : 1);
    std::vector<zc> Mrow(blk_sz);
    const zc itau(0.0, h->tau);
    for (int k = 0; k < c.n_cls; ++k) {
      const zc* Sk = S + k * blk_sz;
      const zc* Hk = H0 + k * blk_sz;
      for (size_t q = 0; q < blk_sz; ++q) Mrow[q] = Sk[q] + itau * Hk[q];
      // entries that point outside the matrix are ignored by contract: zero them so they cannot enter the LU
      for (int i = 0; i < n_rad; ++i)
        for (int d = -w0; d <= w0; ++d)
          if (i + d < 0 || i + d >= n_rad) Mrow[(size_t)i * nd0 + d + w0] = zc(0, 0);
      if (h->path != 0) {
        row_to_col_band_padded(Sk, &Sx[k * blk_p], n_rad, w0, wpad);
        row_to_col_band_padded(Hk, &Hx[k * blk_p], n_rad, w0, wpad);
        row_to_col_band_padded(Mrow.data(), &Mx[k * blk_p], n_rad, w0, wpad);
      } else {
        std::memcpy(&Sx[k * blk_sz], Sk, blk_sz * sizeof(zc));
        std::memcpy(&Hx[k * blk_sz], Hk, blk_sz * sizeof(zc));
        std::memcpy(&Mx[k * blk_sz], Mrow.data(), blk_sz * sizeof(zc));
      }
      double growth = 1.0;
      if (!build_partitioned_factors(Mrow, plan, &Lc[(size_t)k * n_rad * w0], &Uc[(size_t)k * n_rad * (w0 + 1)],
                                     plan.P > 1 ? &Wsp[(size_t)k * n_rad * 2 * w0] : nullptr,
                                     plan.P > 1 ? &Corner[(size_t)k * plan.P * 2 * ww] : nullptr,
                                     plan.P > 1 ? &Schur[(size_t)k * nsep * 3 * ww] : nullptr, &growth))
        return TDDE_ESINGULAR;
      h->lu_growth = std::max(h->lu_growth, growth);
    }
    // The in-iteration applies of the banded path replace the block part by the known right-hand side of the solve (A y = p + ...),
    // which is exact up to the backward error of the unpivoted LU, about eps x growth.  Keep that three orders below rtol.
    h->use_subst = (h->lu_growth * 2.3e-16 <= 1e-3 * c.rtol) && !std::getenv("TDDE_NO_SUBST");
    int rc;
    if ((rc = dev_upload(&h->d_S, reinterpret_cast<cplx*>(Sx.data()), Sx.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_H0, reinterpret_cast<cplx*>(Hx.data()), Hx.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_Mp, reinterpret_cast<cplx*>(Mx.data()), Mx.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_blk_tmp, (cplx*)nullptr, Mx.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_Lcol, reinterpret_cast<cplx*>(Lc.data()), Lc.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_Ucol, reinterpret_cast<cplx*>(Uc.data()), Uc.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_Wsp, reinterpret_cast<cplx*>(Wsp.data()), Wsp.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_Corner, reinterpret_cast<cplx*>(Corner.data()), Corner.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_Schur, reinterpret_cast<cplx*>(Schur.data()), Schur.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_rsm, (cplx*)nullptr, (size_t)plan.P * w0 * h->ld, s))) return rc;
    if ((rc = dev_upload(&h->d_rsp, (cplx*)nullptr, (size_t)plan.P * w0 * h->ld, s))) return rc;
    CU(cudaStreamSynchronize(s));
  }
  // coupling terms
  if (h->path == 1 && T > 0) {
    int nslots = 0;
    for (int L = 0; L < T; ++L) nslots += 2 * (m0 + ms * L);
    std::vector<zc> Aoff((size_t)nslots * h->ld, zc(0, 0));
    int slot0 = 0;
    for (int L = 0; L < T; ++L) {
      const int m = m0 + ms * L;
      const zc* val = reinterpret_cast<const zc*>(terms[L].A_val);
      for (int a = 0; a < c.n_ang; ++a)
        for (int q = terms[L].A_rowptr[a]; q < terms[L].A_rowptr[a + 1]; ++q) {
          const int o = terms[L].A_col[q] - a;
          const int qq = o < 0 ? o + m : m + o - 1;
          Aoff[(size_t)(slot0 + qq) * h->ld + a] = val[q];
        }
      slot0 += 2 * m;
    }
    int rc = dev_upload(&h->d_Aoff, reinterpret_cast<cplx*>(Aoff.data()), Aoff.size(), s);
    if (rc) return rc;
    CU(cudaStreamSynchronize(s));
  }
  {
    // per CTA (128 consecutive channels): the first TDDE_AP_MAXC distinct classes are staged in shared memory
    // (used by the banded apply and by the preconditioner's correction kernel)
    const int n_cta = (h->ld + TDDE_AP_NC - 1) / TDDE_AP_NC;
    std::vector<int> slot(h->ld, -1), cta_cls((size_t)n_cta * TDDE_AP_MAXC, -1);
    int cmax = 0;
    for (int b = 0; b < n_cta; ++b) {
      int cnt = 0;
      for (int a = b * TDDE_AP_NC; a < std::min(h->ld, (b + 1) * TDDE_AP_NC); ++a) {
        const int k = a < c.n_ang ? cls_of_chan[a] : 0;
        int q = 0;
        while (q < cnt && cta_cls[(size_t)b * TDDE_AP_MAXC + q] != k) ++q;
        if (q == cnt && cnt < TDDE_AP_MAXC) cta_cls[(size_t)b * TDDE_AP_MAXC + cnt++] = k;
        slot[a] = q < cnt ? q : -1;
      }
      cmax = std::max(cmax, cnt);
    }
    h->cta_cls_max = std::max(1, cmax);
    int rc;
    if ((rc = dev_upload(&h->d_slot, slot.data(), slot.size(), s))) return rc;
    if ((rc = dev_upload(&h->d_cta_cls, cta_cls.data(), cta_cls.size(), s))) return rc;
    CU(cudaStreamSynchronize(s));
  }
  if (h->path != 0) {
    int rc;
    std::vector<zc> Rall((size_t)n_rad * std::max(T, 1) * ndp), Rc((size_t)n_rad * ndp);
    for (int L = 0; L < T; ++L) {
      row_to_col_band_padded(reinterpret_cast<const zc*>(terms[L].R_band), Rc.data(), n_rad, terms[L].w, wpad);
      for (int j = 0; j < n_rad; ++j)
        std::memcpy(&Rall[((size_t)j * T + L) * ndp], &Rc[(size_t)j * ndp], ndp * sizeof(zc));
    }
    if ((rc = dev_upload(&h->d_Rall, reinterpret_cast<cplx*>(Rall.data()), Rall.size(), s))) return rc;
    // DMMA variant of the in-iteration apply (tdde_apply_mma.cu): fragment table + its own segment length (64-channel CTAs,
    // one per SM, rows in multiples of 8)
    if (h->path == 1 && T > 0 && apply_mma_available(T, h->bM0, h->bMS, h->bW) && !std::getenv("TDDE_NO_MMA")) {
      std::vector<double> frags;
      if (build_mma_frags(T, h->bW, n_rad, Rall.data(), frags)) {
        if ((rc = dev_upload(&h->d_Rfrag, frags.data(), frags.size(), s))) return rc;
        const int nc = apply_mma_channels(h->bW), chan_blocks = (h->ld + nc - 1) / nc, halo = apply_mma_halo(h->bW);
        long long best_cost = -1;
        int best_seg = (n_rad + 7) / 8 * 8;
        for (int seg = 8; seg <= (n_rad + 7) / 8 * 8; seg += 8) {
          const long long ctas = (long long)chan_blocks * ((n_rad + seg - 1) / seg);
          const long long waves = (ctas + h->num_sms - 1) / h->num_sms;
          const long long cost = waves * (seg + halo);
          if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_seg = seg; }
        }
        h->seg_len_m = best_seg;
        if (const char* env = std::getenv("TDDE_MMA_SEG")) h->seg_len_m = std::max(8, std::atoi(env) / 8 * 8);
        // Start of step as block pass + DMMA coupling apply.  Measured on B200 (ms per step, split / one H-apply + S-apply), with the
        // final block pass (at most four classes staged, tensor-map x rows): HBM-scale T = 7, W = 6: 7.85 / 8.01; W = 9: 10.19 / 10.53;
        // Large T = 5: 1.582 / 1.550; Medium T = 5: 0.406 / 0.372.  So: where the register-window kernel needs its two-group term
        // split (T >= 6).  TDDE_SPLIT_START / TDDE_NO_SPLIT_START force it (tests).
        h->split_start = h->use_subst && (T >= 6 || std::getenv("TDDE_SPLIT_START"));
        if (std::getenv("TDDE_NO_SPLIT_START")) h->split_start = false;
      }
    }
    if (h->path == 2) {
      if ((rc = dev_upload(&h->d_spval, reinterpret_cast<cplx*>(ell_val.data()), ell_val.size(), s))) return rc;
      if ((rc = dev_upload(&h->d_spcol, ell_col.data(), ell_col.size(), s))) return rc;
    }
    CU(cudaStreamSynchronize(s));
  }
  for (int L = 0; L < T && h->path == 0; ++L) {
    const int w = terms[L].w, nd = 2 * w + 1;
    h->w[L] = w;
    const zc* R = reinterpret_cast<const zc*>(terms[L].R_band);
    std::vector<zc> Rx((size_t)n_rad * nd);
    std::memcpy(Rx.data(), R, Rx.size() * sizeof(zc));
    int rc;
    if ((rc = dev_upload(&h->d_R[L], reinterpret_cast<cplx*>(Rx.data()), Rx.size(), s))) return rc;
    {
      const int nnz = terms[L].A_rowptr[c.n_ang];
      std::vector<int> rp(h->ld + 1, nnz);
      for (int a = 0; a <= c.n_ang; ++a) rp[a] = terms[L].A_rowptr[a];
      if ((rc = dev_upload(&h->d_Arowptr[L], rp.data(), rp.size(), s))) return rc;
      if ((rc = dev_upload(&h->d_Acol[L], terms[L].A_col, (size_t)nnz, s))) return rc;
      if ((rc = dev_upload(&h->d_Aval[L], reinterpret_cast<const cplx*>(terms[L].A_val), (size_t)nnz, s))) return rc;
    }
    CU(cudaStreamSynchronize(s));
  }
  // work vectors
  cplx** vecs[] = {&h->X, &h->r, &h->rhat, &h->p, &h->v, &h->s, &h->t, &h->y, &h->z};
  for (cplx** v : vecs) {
    CU(cudaMalloc((void**)v, (size_t)h->nint * sizeof(cplx)));
    CU(cudaMemsetAsync(*v, 0, (size_t)h->nint * sizeof(cplx), s));
  }
  // 2-D tensor maps of the work vectors ([n_rad][2 ld] doubles, box = 128 channels x TDDE_AP_JC rows): the S-only
  // apply fetches its x tile with one tensor TMA copy per stage instead of one bulk copy per row.  Optional: if the
  // driver entry point or the encoding is unavailable the kernel keeps using 1-D bulk copies.
  h->have_xmaps = false;
  if (h->path == 1 && h->ld >= 128) {
    typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess && fn &&
        qres == cudaDriverEntryPointSuccess) {
      bool ok = true;
      int q = 0;
      for (cplx** v : vecs) {
        const cuuint64_t gdim[2] = {(cuuint64_t)2 * h->ld, (cuuint64_t)n_rad};
        const cuuint64_t gstride[1] = {(cuuint64_t)h->ld * sizeof(cplx)};
        const cuuint32_t box[2] = {256, TDDE_AP_JC};
        const cuuint32_t estr[2] = {1, 1};
        ok = ok && ((encode_fn)fn)(&h->xmaps[q++], CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, *v, gdim, gstride, box, estr,
                                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
      }
      h->have_xmaps = ok && !std::getenv("TDDE_NO_XMAP");
    }
    cudaGetLastError();
  }
  // state and scratch
  CU(cudaMalloc((void**)&h->d_st, sizeof(SolverState)));
  CU(cudaMalloc((void**)&h->d_st_bench, sizeof(SolverState)));
  CU(cudaMallocHost((void**)&h->h_st, sizeof(SolverState)));
  std::memset(h->h_st, 0, sizeof(SolverState));
  h->h_st->rtol2 = c.rtol * c.rtol;
  h->h_st->max_half = 2 * c.max_iter;
  h->h_st->done = 1;
  CU(cudaMemcpyAsync(h->d_st, h->h_st, sizeof(SolverState), cudaMemcpyHostToDevice, s));
  CU(cudaStreamSynchronize(s));
  {
    SolverState b;
    std::memset(&b, 0, sizeof(b));
    b.rho = b.rho_old = b.alpha = b.omega = b.beta = make_double2(1.0, 0.0);
    b.force = 1; b.max_half = 1 << 30; b.nb2 = 1.0;
    CU(cudaMemcpy(h->d_st_bench, &b, sizeof(b), cudaMemcpyHostToDevice));
  }
  CU(cudaMalloc((void**)&h->d_partials, (size_t)TDDE_MAX_PARTIAL_BLOCKS * 4 * sizeof(double)));
  CU(cudaMalloc((void**)&h->d_ticket, sizeof(unsigned int)));
  CU(cudaMemsetAsync(h->d_ticket, 0, sizeof(unsigned int), s));
  const size_t tcount = T > 0 ? T : 1;
  CU(cudaMalloc((void**)&h->d_g_small, tcount * sizeof(double)));
  CU(cudaMalloc((void**)&h->d_zero_g, tcount * sizeof(double)));
  CU(cudaMemsetAsync(h->d_zero_g, 0, tcount * sizeof(double), s));
  CU(cudaMemsetAsync(h->d_g_small, 0, tcount * sizeof(double), s));
  CU(cudaStreamSynchronize(s));
  return 0;
}

extern "C" int tdde_create(tdde_handle** out, const tdde_config* cfg, const tdde_c64* S_band, const tdde_c64* H0_band,
                           const int32_t* cls_of_chan, const tdde_term* terms, void* cuda_stream) {
  if (!out) return TDDE_EINVAL;
  *out = nullptr;
  int rc = validate(cfg, S_band, H0_band, cls_of_chan, terms);
  if (rc) return rc;
  int ndev = 0;
  CU(cudaGetDeviceCount(&ndev));
  if (ndev <= 0) { g_last_cuda_error = "no CUDA device"; return TDDE_ECUDA; }
  tdde_handle* h = new (std::nothrow) tdde_handle();
  if (!h) return TDDE_ENOMEM;
  h->cfg = *cfg;
  h->stream = (cudaStream_t)cuda_stream;
  try {
    rc = create_impl(h, S_band, H0_band, cls_of_chan, terms);
  } catch (const std::bad_alloc&) {
    rc = TDDE_ENOMEM;
  } catch (...) {
    rc = TDDE_EINVAL;
  }
  if (rc) { tdde_destroy(h); return rc; }
  *out = h;
  return 0;
}
