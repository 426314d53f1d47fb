// Warp-level tridiagonal solve and the Fisher-KPP level matrix (shared by the classic and the fused 1D kernels).
#pragma once
#include "device_utils.cuh"
#include "snap_internal.h"

namespace snap {

// (pivots of the diagonally dominant SPD level matrices are positive and of order one: reciprocals by rcp_pos)
// ------------------------------------------------------------------------------------------------
// warp tridiagonal solve (Fisher): rows owned contiguously, Q per lane; partition method —
// each lane eliminates its Q-1 interior unknowns against its own last unknown (the separator) and the
// previous lane's, the 32 separators are solved by parallel cyclic reduction with shuffles.
// Row j of lane p:  a[j] x_{-1} + b[j] x_j + c[j] x_{+1} = d[j].  a of the first global row and c of the
// last must be 0; padding rows are identity rows.  Solution returned in d.
// ------------------------------------------------------------------------------------------------
template <int Q>
__device__ __forceinline__ void warp_tridiag(const double (&a)[Q], const double (&b)[Q], const double (&c)[Q],
                                             double (&d)[Q], int lane) {
  double ra, rb, rc, rd;
  double v[Q], al[Q], be[Q];
  if (Q > 1) {
    double cp[Q];
    {
      const double inv = rcp_pos(b[0]);
      cp[0] = (Q > 2 ? c[0] : 0.0) * inv;
      v[0] = d[0] * inv;
      al[0] = a[0] * inv;
      be[0] = (Q == 2 ? c[0] : 0.0) * inv;
    }
#pragma unroll
    for (int j = 1; j < Q - 1; ++j) {
      const double inv = rcp_pos(b[j] - a[j] * cp[j - 1]);
      cp[j] = (j < Q - 2 ? c[j] : 0.0) * inv;
      v[j] = (d[j] - a[j] * v[j - 1]) * inv;
      al[j] = (-a[j] * al[j - 1]) * inv;
      be[j] = ((j == Q - 2 ? c[j] : 0.0) - a[j] * be[j - 1]) * inv;
    }
#pragma unroll
    for (int j = Q - 3; j >= 0; --j) {
      v[j] -= cp[j] * v[j + 1];
      al[j] -= cp[j] * al[j + 1];
      be[j] -= cp[j] * be[j + 1];
    }
    // separator row Q-1: a x_{Q-2} + b s_p + c x_{p+1,0} = d with x = v - s_{p-1} al - s_p be
    const double v0n = __shfl_down_sync(SNAP_FULL, v[0], 1);
    const double al0n = __shfl_down_sync(SNAP_FULL, al[0], 1);
    const double be0n = __shfl_down_sync(SNAP_FULL, be[0], 1);
    const double cl = (lane == 31) ? 0.0 : c[Q - 1];
    ra = -a[Q - 1] * al[Q - 2];
    rb = b[Q - 1] - a[Q - 1] * be[Q - 2] - cl * al0n;
    rc = -cl * be0n;
    rd = d[Q - 1] - a[Q - 1] * v[Q - 2] - cl * v0n;
  } else {
    ra = a[0];
    rb = b[0];
    rc = (lane == 31) ? 0.0 : c[0];
    rd = d[0];
  }
  if (lane == 0) ra = 0.0;
  // parallel cyclic reduction over the 32 lanes, rows kept normalised (rb == 1)
  {
    const double inv = rcp_pos(rb);
    ra *= inv;
    rc *= inv;
    rd *= inv;
  }
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) {
    double alo = __shfl_up_sync(SNAP_FULL, ra, s), clo = __shfl_up_sync(SNAP_FULL, rc, s),
           dlo = __shfl_up_sync(SNAP_FULL, rd, s);
    double ahi = __shfl_down_sync(SNAP_FULL, ra, s), chi = __shfl_down_sync(SNAP_FULL, rc, s),
           dhi = __shfl_down_sync(SNAP_FULL, rd, s);
    if (lane < s) { alo = 0.0; clo = 0.0; dlo = 0.0; }
    if (lane + s > 31) { ahi = 0.0; chi = 0.0; dhi = 0.0; }
    const double nb = 1.0 - clo * ra - ahi * rc;
    const double inv = rcp_pos(nb);
    const double nd = (rd - dlo * ra - dhi * rc) * inv;
    const double na = (-alo * ra) * inv;
    const double nc = (-chi * rc) * inv;
    ra = na; rc = nc; rd = nd;
  }
  const double s_me = rd;
  if (Q > 1) {
    double s_prev = __shfl_up_sync(SNAP_FULL, s_me, 1);
    if (lane == 0) s_prev = 0.0;
#pragma unroll
    for (int j = 0; j < Q - 1; ++j) d[j] = v[j] - s_prev * al[j] - s_me * be[j];
  }
  d[Q - 1] = s_me;
}

// The same solve for a matrix whose off-diagonal entries are all `off` (0 outside the first / last global row) and whose 32 Q
// rows fill the warp exactly: the two coefficient arrays of the general routine are then two scalars per lane, which is
// 32 registers less in the fused Fisher passes (kernels_1d_fused.cuh).  Same operations on the same values.
template <int Q>
__device__ __forceinline__ void warp_tridiag_sym(const double off, const double (&b)[Q], double (&d)[Q], int lane) {
  const double a0 = (lane == 0) ? 0.0 : off;          // a of the lane's first row
  const double cl = (lane == 31) ? 0.0 : off;         // c of the lane's last row
  double ra, rb, rc, rd;
  double v[Q], al[Q], be[Q];
  if (Q > 1) {
    double cp[Q];
    {
      const double inv = rcp_pos(b[0]);
      cp[0] = (Q > 2 ? off : 0.0) * inv;
      v[0] = d[0] * inv;
      al[0] = a0 * inv;
      be[0] = (Q == 2 ? off : 0.0) * inv;
    }
#pragma unroll
    for (int j = 1; j < Q - 1; ++j) {
      const double inv = rcp_pos(b[j] - off * cp[j - 1]);
      cp[j] = (j < Q - 2 ? off : 0.0) * inv;
      v[j] = (d[j] - off * v[j - 1]) * inv;
      al[j] = (-off * al[j - 1]) * inv;
      be[j] = ((j == Q - 2 ? off : 0.0) - off * be[j - 1]) * inv;
    }
#pragma unroll
    for (int j = Q - 3; j >= 0; --j) {
      v[j] -= cp[j] * v[j + 1];
      al[j] -= cp[j] * al[j + 1];
      be[j] -= cp[j] * be[j + 1];
    }
    const double v0n = __shfl_down_sync(SNAP_FULL, v[0], 1);
    const double al0n = __shfl_down_sync(SNAP_FULL, al[0], 1);
    const double be0n = __shfl_down_sync(SNAP_FULL, be[0], 1);
    ra = -off * al[Q - 2];
    rb = b[Q - 1] - off * be[Q - 2] - cl * al0n;
    rc = -cl * be0n;
    rd = d[Q - 1] - off * v[Q - 2] - cl * v0n;
  } else {
    ra = a0;
    rb = b[0];
    rc = cl;
    rd = d[0];
  }
  if (lane == 0) ra = 0.0;
  {
    const double inv = rcp_pos(rb);
    ra *= inv;
    rc *= inv;
    rd *= inv;
  }
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) {
    double alo = __shfl_up_sync(SNAP_FULL, ra, s), clo = __shfl_up_sync(SNAP_FULL, rc, s),
           dlo = __shfl_up_sync(SNAP_FULL, rd, s);
    double ahi = __shfl_down_sync(SNAP_FULL, ra, s), chi = __shfl_down_sync(SNAP_FULL, rc, s),
           dhi = __shfl_down_sync(SNAP_FULL, rd, s);
    if (lane < s) { alo = 0.0; clo = 0.0; dlo = 0.0; }
    if (lane + s > 31) { ahi = 0.0; chi = 0.0; dhi = 0.0; }
    const double nb = 1.0 - clo * ra - ahi * rc;
    const double inv = rcp_pos(nb);
    const double nd = (rd - dlo * ra - dhi * rc) * inv;
    const double na = (-alo * ra) * inv;
    const double nc = (-chi * rc) * inv;
    ra = na; rc = nc; rd = nd;
  }
  const double s_me = rd;
  if (Q > 1) {
    double s_prev = __shfl_up_sync(SNAP_FULL, s_me, 1);
    if (lane == 0) s_prev = 0.0;
#pragma unroll
    for (int j = 0; j < Q - 1; ++j) d[j] = v[j] - s_prev * al[j] - s_me * be[j];
  }
  d[Q - 1] = s_me;
}

// Fisher: tridiagonal T_k = I - dt D Lap_h - dt rho diag(1 - 2u) restricted to this lane's rows.
template <int Q>
__device__ __forceinline__ void fisher_matrix(const DevParams& P, const double (&uk)[Q], int lane, double (&a)[Q],
                                              double (&b)[Q], double (&c)[Q]) {
#pragma unroll
  for (int j = 0; j < Q; ++j) {
    const int i = lane * Q + j;
    if (i < P.nx) {
      const double nnb = (i == 0 || i == P.nx - 1) ? 1.0 : 2.0;
      a[j] = (i == 0) ? 0.0 : -P.fi_a;
      c[j] = (i == P.nx - 1) ? 0.0 : -P.fi_a;
      b[j] = 1.0 + P.fi_a * nnb - P.fi_dtrho * (1.0 - 2.0 * uk[j]);
    } else {
      a[j] = 0.0; b[j] = 1.0; c[j] = 0.0;
    }
  }
}

// diagonal of that matrix for a warp whose 32 Q rows are the whole level (the off-diagonals are -fa)
template <int Q>
__device__ __forceinline__ void fisher_diag(double fa, double fr, const double (&uk)[Q], int lane, double (&b)[Q]) {
#pragma unroll
  for (int c = 0; c < Q; ++c) {
    const double nnb = ((lane == 0 && c == 0) || (lane == 31 && c == Q - 1)) ? 1.0 : 2.0;
    b[c] = 1.0 + fa * nnb - fr * (1.0 - 2.0 * uk[c]);
  }
}

}  // namespace snap
