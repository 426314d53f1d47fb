// Float32 / tolerance 1e-5 mode ("single-precision floating-point values (Float32) ... convergence tolerance
// fixed to 1e-5") for the Burgers family (kinds 1, 4), multiplier-free (PCFM's pull-back uses u_1 only,
// Eq. 3).  Same method as kernels_1d_fused.cuh -- forward passes that carry JT Gauss-Newton iterations per level,
//     q_0 = h_0 ,  q_k = h_k + A_{k-1} q_{k-1} ,  x+ = x - q     (J_loc square: the step is Newton on h) --
// in fp32: one warp per sample, lane l owns the Q contiguous cells l Q .., rows move as plain coalesced 128-bit loads with the
// next level prefetched in registers (a 256-cell row is 1 KB: no shared-memory staging is needed), neighbours by shuffles.
// A pass runs JT - 1 updates and evaluates ||h||_inf at every iterate it visits (local rows and, kind 4, the mass rows);
// the sample is done when an iterate met tol and at least `polish` more steps followed it.  Full steps only (the merit
// test is dormant on these row sets, R17): a step after which ||h||_inf grows ends the sample with status -2.
#pragma once
#include "device_utils.cuh"
#include "snap_internal.h"

namespace snap {

struct ProjF32Args {
  DevParams P;
  int batch;
  const float* u_hat;
  const float* cdata;
  float* u_star;
  int* iters;
  float* bufA;   // [batch][n]
  float* bufB;
  float tol;
};

template <int Q>
__device__ __forceinline__ void ldrow_f32(const float* __restrict__ g, float (&x)[Q]) {
  if constexpr (Q >= 4) {
#pragma unroll
    for (int c = 0; c < Q / 4; ++c) {
      const float4 t = reinterpret_cast<const float4*>(g)[c];
      x[4 * c] = t.x; x[4 * c + 1] = t.y; x[4 * c + 2] = t.z; x[4 * c + 3] = t.w;
    }
  } else {
#pragma unroll
    for (int c = 0; c < Q; ++c) x[c] = g[c];
  }
}
template <int Q>
__device__ __forceinline__ void strow_f32(float* __restrict__ g, const float (&x)[Q]) {
  if constexpr (Q >= 4) {
#pragma unroll
    for (int c = 0; c < Q / 4; ++c) reinterpret_cast<float4*>(g)[c] = make_float4(x[4 * c], x[4 * c + 1], x[4 * c + 2], x[4 * c + 3]);
  } else {
#pragma unroll
    for (int c = 0; c < Q; ++c) g[c] = x[c];
  }
}
__device__ __forceinline__ float wmaxf(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(SNAP_FULL, v, o));
  return v;
}
__device__ __forceinline__ float wsumf(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(SNAP_FULL, v, o);
  return v;
}

// One forward pass: T = NU + 1 iterations per level (NU updates, then the evaluation of the last iterate); reads x, writes
// the iterate x_NU to `xo` (NU > 0).  hmax[t] = ||h(x_t)||_inf, t = 0..NU (warp-uniform on return).
template <int Q, int JT>
__device__ __forceinline__ void f32_pass(const DevParams& P, int lane, const float* __restrict__ x, const float* __restrict__ u0,
                                         float* __restrict__ xo, int NU, float M0, float (&hmax)[JT]) {
  constexpr int nx = 32 * Q;
  const int nt = P.nt, first = lane * Q;
  const float a0 = (float)P.bs_a0, e = (float)P.bs_e, qs = (float)P.bs_qs, hs = (float)P.bs_hs, dxm = (float)P.dx;
  const bool has_mass = P.has_mass != 0;
  float phi[JT][Q], cc[JT][Q];
  {
    float u0r[Q];
    ldrow_f32<Q>(u0 + first, u0r);
#pragma unroll
    for (int t = 0; t < JT; ++t) {
#pragma unroll
      for (int c = 0; c < Q; ++c) { phi[t][c] = u0r[c]; cc[t][c] = 0.f; }
      hmax[t] = 0.f;
    }
  }
  float vn[Q];
  ldrow_f32<Q>(x + first, vn);
  for (int k = 0; k < nt; ++k) {
    float v[Q];
#pragma unroll
    for (int c = 0; c < Q; ++c) v[c] = vn[c];
    if (k + 1 < nt) ldrow_f32<Q>(x + (size_t)(k + 1) * nx + first, vn);    // next level travels during this one
    float msum[JT];
#pragma unroll
    for (int t = 0; t < JT; ++t) msum[t] = 0.f;
    float vL = 0.f, vR = 0.f;
#pragma unroll
    for (int t = 0; t < JT; ++t) {
      if (t <= NU) {
        float q[Q], hm = 0.f, ms = 0.f;
#pragma unroll
        for (int c = 0; c < Q; ++c) {
          const float h = v[c] - phi[t][c];
          q[c] = h + cc[t][c];
          hm = fmaxf(hm, fabsf(h));
          ms += v[c];
        }
        msum[t] = ms;                        // mass row of this level and iterate: reduced after the iterations
        hmax[t] = fmaxf(hmax[t], hm);
        // the neighbours' end cells: exchanged for the first iterate of a level, then updated like the neighbour updates them
        if (t == 0) { vL = __shfl_sync(SNAP_FULL, v[Q - 1], (lane + 31) & 31); vR = __shfl_sync(SNAP_FULL, v[0], (lane + 1) & 31); }
        const float qL = __shfl_sync(SNAP_FULL, q[Q - 1], (lane + 31) & 31), qR = __shfl_sync(SNAP_FULL, q[0], (lane + 1) & 31);
        float um = vL, ql = qL;
#pragma unroll
        for (int c = 0; c < Q; ++c) {
          const float up = (c < Q - 1) ? v[c + 1] : vR, qr = (c < Q - 1) ? q[c + 1] : qR;
          const float vc = v[c], qc = q[c];
          phi[t][c] = fmaf(a0, vc, (up + um) * fmaf(-qs, up - um, e));
          cc[t][c] = fmaf(fmaf(-hs, up, e), qr, fmaf(fmaf(hs, um, e), ql, a0 * qc));
          um = vc; ql = qc;
          if (t < NU) v[c] = vc - qc;
        }
        if (t < NU) { vL -= qL; vR -= qR; }
      }
    }
    if (NU > 0) strow_f32<Q>(xo + (size_t)k * nx + first, v);
    if (has_mass) {     // JT interleaved butterflies, off the critical path of the level recurrence
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int t = 0; t < JT; ++t) msum[t] += __shfl_xor_sync(SNAP_FULL, msum[t], o);
      }
#pragma unroll
      for (int t = 0; t < JT; ++t)
        if (t <= NU) hmax[t] = fmaxf(hmax[t], fabsf(fmaf(dxm, msum[t], -M0)));
    }
  }
#pragma unroll
  for (int t = 0; t < JT; ++t) hmax[t] = wmaxf(hmax[t]);
}

// The same pass with packed fp32 arithmetic (sm_100: add / mul / fma on float2, one instruction for two cells): the pass
// is bound by instruction issue (one warp per sample, two warps per scheduler), and a packed instruction does the work of
// two.  A lane pairs cell c with cell c + Q/2 of its Q contiguous cells, so that the right / left neighbours of pair c are
// the pairs c + 1 / c - 1 (aligned register pairs); only the first and the last pair take one component from the
// neighbouring lane.  Phi is carried negated (h = x + (-Phi)): negations are exact, the results equal the scalar pass bit
// for bit except for the order of the mass-row sums.
template <int Q, int JT>
__device__ __forceinline__ void f32_pass_x2(const DevParams& P, int lane, const float* __restrict__ x,
                                            const float* __restrict__ u0, float* __restrict__ xo, int NU, float M0,
                                            float (&hmax)[JT]) {
  static_assert(Q >= 2 && Q % 2 == 0, "pairs of cells");
  constexpr int nx = 32 * Q, H = Q / 2;
  const int nt = P.nt, first = lane * Q;
  const float a0 = (float)P.bs_a0, e = (float)P.bs_e, qs = (float)P.bs_qs, hs = (float)P.bs_hs, dxm = (float)P.dx;
  const float2 A0 = make_float2(a0, a0), NA0 = make_float2(-a0, -a0), E2 = make_float2(e, e), NE2 = make_float2(-e, -e);
  const float2 QS = make_float2(qs, qs), HS = make_float2(hs, hs), NHS = make_float2(-hs, -hs), M1 = make_float2(-1.f, -1.f);
  const bool has_mass = P.has_mass != 0;
  float2 nphi[JT][H], cc[JT][H];
  {
    float u0r[Q];
    ldrow_f32<Q>(u0 + first, u0r);
#pragma unroll
    for (int t = 0; t < JT; ++t) {
#pragma unroll
      for (int c = 0; c < H; ++c) { nphi[t][c] = make_float2(-u0r[c], -u0r[c + H]); cc[t][c] = make_float2(0.f, 0.f); }
      hmax[t] = 0.f;
    }
  }
  float vn[Q];
  ldrow_f32<Q>(x + first, vn);
  for (int k = 0; k < nt; ++k) {
    float2 v[H];
#pragma unroll
    for (int c = 0; c < H; ++c) v[c] = make_float2(vn[c], vn[c + H]);
    if (k + 1 < nt) ldrow_f32<Q>(x + (size_t)(k + 1) * nx + first, vn);    // next level travels during this one
    float msum[JT];
#pragma unroll
    for (int t = 0; t < JT; ++t) msum[t] = 0.f;
    float vL = 0.f, vR = 0.f;            // the neighbours' end cells, carried through the iterations of the level
#pragma unroll
    for (int t = 0; t < JT; ++t) {
      if (t <= NU) {
        float2 q[H], ms = make_float2(0.f, 0.f);
        float hm = 0.f;
#pragma unroll
        for (int c = 0; c < H; ++c) {
          const float2 h = __fadd2_rn(v[c], nphi[t][c]);
          q[c] = __fadd2_rn(h, cc[t][c]);
          hm = fmaxf(hm, fmaxf(fabsf(h.x), fabsf(h.y)));
          ms = __fadd2_rn(ms, v[c]);
        }
        msum[t] = ms.x + ms.y;
        hmax[t] = fmaxf(hmax[t], hm);
        if (t == 0) { vL = __shfl_sync(SNAP_FULL, v[H - 1].y, (lane + 31) & 31); vR = __shfl_sync(SNAP_FULL, v[0].x, (lane + 1) & 31); }
        const float qL = __shfl_sync(SNAP_FULL, q[H - 1].y, (lane + 31) & 31), qR = __shfl_sync(SNAP_FULL, q[0].x, (lane + 1) & 31);
        // pair c = (cell c, cell c + H): left neighbours (c - 1, c + H - 1), right neighbours (c + 1, c + H + 1)
        const float2 vLo = make_float2(vL, v[H - 1].x), vHi = make_float2(v[0].y, vR);
        const float2 qLo = make_float2(qL, q[H - 1].x), qHi = make_float2(q[0].y, qR);
        float2 nph[H], ccn[H];
#pragma unroll
        for (int c = 0; c < H; ++c) {
          const float2 um = (c > 0) ? v[c > 0 ? c - 1 : 0] : vLo, up = (c < H - 1) ? v[c < H - 1 ? c + 1 : 0] : vHi;
          const float2 ql = (c > 0) ? q[c > 0 ? c - 1 : 0] : qLo, qr = (c < H - 1) ? q[c < H - 1 ? c + 1 : 0] : qHi;
          const float2 sum = __fadd2_rn(up, um), dif = __ffma2_rn(um, M1, up);
          const float2 w = __ffma2_rn(QS, dif, NE2);                                   // -(e - qs (up - um))
          nph[c] = __ffma2_rn(NA0, v[c], __fmul2_rn(sum, w));                          // -Phi
          ccn[c] = __ffma2_rn(__ffma2_rn(NHS, up, E2), qr, __ffma2_rn(__ffma2_rn(HS, um, E2), ql, __fmul2_rn(A0, q[c])));
        }
#pragma unroll
        for (int c = 0; c < H; ++c) {
          nphi[t][c] = nph[c];
          cc[t][c] = ccn[c];
          if (t < NU) v[c] = __ffma2_rn(q[c], M1, v[c]);
        }
        if (t < NU) { vL = fmaf(qL, -1.f, vL); vR = fmaf(qR, -1.f, vR); }   // as the neighbour updates them (same fma)
      }
    }
    if (NU > 0) {
      float vo[Q];
#pragma unroll
      for (int c = 0; c < H; ++c) { vo[c] = v[c].x; vo[c + H] = v[c].y; }
      strow_f32<Q>(xo + (size_t)k * nx + first, vo);
    }
    if (has_mass) {     // JT interleaved butterflies, off the critical path of the level recurrence
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int t = 0; t < JT; ++t) msum[t] += __shfl_xor_sync(SNAP_FULL, msum[t], o);
      }
#pragma unroll
      for (int t = 0; t < JT; ++t)
        if (t <= NU) hmax[t] = fmaxf(hmax[t], fabsf(fmaf(dxm, msum[t], -M0)));
    }
  }
#pragma unroll
  for (int t = 0; t < JT; ++t) hmax[t] = wmaxf(hmax[t]);
}

template <int Q, int JT>
__global__ void __launch_bounds__(256) project1d_f32_kernel(const __grid_constant__ ProjF32Args A) {
  const DevParams& P = A.P;
  const int lane = threadIdx.x & 31;
  const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (b >= A.batch) return;
  constexpr int nx = 32 * Q;
  const size_t n = (size_t)P.n;
  const float* uh = A.u_hat + (size_t)b * n;
  const float* u0 = A.cdata + (size_t)b * nx;
  float* ustar = A.u_star + (size_t)b * n;
  float* bufA = A.bufA + (size_t)b * n;
  float* bufB = A.bufB + (size_t)b * n;
  float M0 = 0.f;
  if (P.has_mass) {
    float s = 0.f;
    for (int i = lane; i < nx; i += 32) s += u0[i];
    M0 = (float)P.dx * wsumf(s);
  }
  const float tol = A.tol;
  // iterates ping-pong between bufA and u_star itself (bufB when u_star aliases u_hat): the usual two passes (JT - 1
  // updates; then the remaining polish step) end in u_star and need no copy
  float* const alt = (ustar != uh) ? ustar : bufB;
  const float* cur = uh;
  int steps = 0, lin = 0, status = 0, since = -1;     // since: steps taken after the first iterate that met tol (-1: none yet)
  float hprev = 3.4e38f;
  bool done = false, first_pass = true;
  while (!done) {
    float* xo = (cur == bufA) ? alt : bufA;
    int NU = JT - 1;
    if (since >= 0 && P.polish - since < NU) NU = P.polish - since;   // only the remaining polish steps
    if (NU > P.max_iter - steps && since < 0) NU = P.max_iter - steps;
    if (NU < 0) NU = 0;
    float hmax[JT];
    if constexpr (Q >= 2) f32_pass_x2<Q, JT>(P, lane, cur, u0, xo, NU, M0, hmax);
    else f32_pass<Q, JT>(P, lane, cur, u0, xo, NU, M0, hmax);
    __syncwarp();
    // walk the iterates x_0 .. x_NU of this pass (x_0 of a later pass was judged as the last iterate of the previous one)
    if (!first_pass && NU > 0) { ++steps; if (since >= 0) ++since; }   // the step x_0 -> x_1 of a later pass
    for (int t = first_pass ? 0 : 1; t <= NU; ++t) {
      const float hv = hmax[t];
      ++lin;
      if (!(hv <= 3.4e38f)) { status = SNAP_ST_NONFINITE; done = true; break; }
      if (since < 0) {
        if (hv < tol) since = 0;
        else if (hv > hprev && t > 0) { status = SNAP_ST_LINESEARCH; done = true; break; }   // a full step that does not descend
      }
      hprev = hv;
      if (t < NU) { ++steps; if (since >= 0) ++since; }
    }
    first_pass = false;
    if (done) break;
    if (NU > 0) cur = xo;
    if (since >= P.polish) done = true;                       // converged and polished: cur is final
    else if (since < 0 && steps >= P.max_iter) { status = SNAP_ST_MAXITER; done = true; }
  }
  // u* <- final iterate (u_hat on a non-finite sample, R16)
  const float* fin = (status == SNAP_ST_NONFINITE) ? uh : cur;
  if (fin != ustar) {   // 128-bit stream, 8 loads in flight per lane
    const float4* s4 = reinterpret_cast<const float4*>(fin);
    float4* d4 = reinterpret_cast<float4*>(ustar);
    const size_t n4 = n / 4;
    size_t i = lane;
    for (; i + 7 * 32 < n4; i += 8 * 32) {
      float4 t[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) t[u] = s4[i + u * 32];
#pragma unroll
      for (int u = 0; u < 8; ++u) d4[i + u * 32] = t[u];
    }
    for (; i < n4; i += 32) d4[i] = s4[i];
  }
  if (lane == 0) A.iters[b] = (status == 0) ? lin : status;
}

}  // namespace snap
