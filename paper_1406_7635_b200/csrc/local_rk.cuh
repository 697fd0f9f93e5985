// local_rk.cuh - local field terms, Landau-Lifshitz torque and the Dormand-Prince stage kernels.
#pragma once
#include "common.cuh"

__device__ __forceinline__ int tri_index(int a, int b) {  // lower-triangular table index (Fig. 1, L31)
  int i = max(a, b), j = min(a, b);
  return i * (i + 1) / 2 + j;
}

// Standard normal eta(seed, component, counter) of the thermal field (Eq. 24): the counter-based generator
// of synth/rng.py restated (splitmix64 finaliser over seed, stream, index; 53-bit uniforms; Box-Muller)
// in fp64, so that both sides draw the same numbers.
__device__ __forceinline__ unsigned long long mm_mix64(unsigned long long z) {
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}
__device__ __forceinline__ double mm_uniform01(unsigned long long seed, unsigned long long stream, unsigned long long index) {
  unsigned long long z = mm_mix64(seed + 0x9E3779B97F4A7C15ull);
  z = mm_mix64(z ^ (stream * 0xD1B54A32D192ED03ull));
  z = mm_mix64(z + index * 0x9E3779B97F4A7C15ull);
  return (double)(z >> 11) * (1.0 / 9007199254740992.0);
}
__device__ __forceinline__ float mm_eta(unsigned long long seed, int comp, unsigned long long index) {
  const double u1 = mm_uniform01(seed, comp, index), u2 = mm_uniform01(seed, 3 + comp, index);
  return (float)(sqrt(-2.0 * log(1.0 - u1)) * cospi(2.0 * u2));
}

// Heisenberg + Dzyaloshinskii-Moriya exchange field of ONE cell with the boundary conditions of Eq. 11-15
// (PAPER.md L215-L257): B_DM = (2D/Msat)(dm_z/dx, dm_z/dy, -dm_x/dx - dm_y/dy) by central differences (L246);
// a missing neighbour - outside an open box or a vacuum cell (Msat = 0) - is the virtual
// m + (dm/di)|_dV Delta_i n, and with D != 0 the same virtual neighbour enters Eq. 6 (L248).
// Adds to (bx, by, bz). Used by the local kernels and the energy kernel when a DM strength is set.
__device__ __forceinline__ void exch_dmi_cell(const Geometry& g, const uint8_t* __restrict__ regions, const Luts* __restrict__ lut,
                                              const float* __restrict__ m, long long i, int x, int y, int z, int r, float mx,
                                              float my, float mz, float& bx, float& by, float& bz) {
  const long long N = g.N;
  const float bc = lut->dmi_bc[r], cD = lut->dmi[r], own = __ldg(&lut->exch[tri_index(r, r)]);
  float ex = 0.f, ey = 0.f, ez = 0.f;
  // neighbour at sign = +-1 along axis (0 = x, 1 = y, 2 = z): (nx, ny, nz) and its exchange contribution
  auto nbr = [&](bool inside, long long j, int axis, float sgn, float d, float w, float& nx, float& ny, float& nz) {
    const int rj = inside ? (int)regions[j] : r;
    if (inside && lut->live[rj] > 0.f) {
      nx = m[j]; ny = m[N + j]; nz = m[2 * N + j];
      w *= __ldg(&lut->exch[tri_index(r, rj)]);
    } else {
      const float s = sgn * d * bc;
      nx = mx; ny = my; nz = mz;
      if (axis == 0) { nx = mx - s * mz; nz = mz + s * mx; }
      else if (axis == 1) { ny = my - s * mz; nz = mz + s * my; }
      w *= own;
    }
    ex += w * (nx - mx); ey += w * (ny - my); ez += w * (nz - mz);
  };
  float px, py, pz, qx, qy, qz;
  if (g.Nx > 1) {
    const bool up = x + 1 < g.Nx || g.pbc[0], dn = x > 0 || g.pbc[0];
    nbr(up, x + 1 < g.Nx ? i + 1 : i + 1 - g.Nx, 0, 1.f, g.dx, g.inv_dx2, px, py, pz);
    nbr(dn, x > 0 ? i - 1 : i - 1 + g.Nx, 0, -1.f, g.dx, g.inv_dx2, qx, qy, qz);
    const float h = cD / (2.f * g.dx);
    bx += h * (pz - qz); bz -= h * (px - qx);
  }
  if (g.Ny > 1) {
    const long long s = g.Nx;
    const bool up = y + 1 < g.Ny || g.pbc[1], dn = y > 0 || g.pbc[1];
    nbr(up, y + 1 < g.Ny ? i + s : i + s - s * g.Ny, 1, 1.f, g.dy, g.inv_dy2, px, py, pz);
    nbr(dn, y > 0 ? i - s : i - s + s * g.Ny, 1, -1.f, g.dy, g.inv_dy2, qx, qy, qz);
    const float h = cD / (2.f * g.dy);
    by += h * (pz - qz); bz -= h * (py - qy);
  }
  if (g.Nz > 1) {
    const long long s = (long long)g.Nx * g.Ny;
    const bool up = z + 1 < g.Nz || g.pbc[2], dn = z > 0 || g.pbc[2];
    nbr(up, z + 1 < g.Nz ? i + s : i + s - s * g.Nz, 2, 1.f, 0.f, g.inv_dz2, px, py, pz);
    nbr(dn, z > 0 ? i - s : i - s + s * g.Nz, 2, -1.f, 0.f, g.inv_dz2, qx, qy, qz);
  }
  bx += ex; by += ey; bz += ez;
}

// B_eff = [B_demag] + B_exch (Eq. 6 / Eq. 9) + B_anis (Eq. 18, 21) + B_ext, then either stored as the
// field (out_torque = 0) or turned into the torque over gamma (Eq. 2, sign reading DESIGN.md #5).
// One thread per cell; x fastest so every global access of a warp is one contiguous segment.
__global__ void k_local(Geometry g, const uint8_t* __restrict__ regions, const Luts* __restrict__ lut, DevState* st,
                        int m_role, int bd_role, int dst_role, unsigned mask, int out_torque) {
  if (st->skip) return;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= g.N) return;
  const float* __restrict__ m = st->ptr[m_role];
  const float* __restrict__ bd = st->ptr[bd_role];
  float* __restrict__ dst = st->ptr[dst_role];
  const long long N = g.N;
  const int x = (int)(i % g.Nx);
  const long long t = i / g.Nx;
  const int y = (int)(t % g.Ny), z = (int)(t / g.Ny);
  const int r = regions[i];
  const float mx = m[i], my = m[N + i], mz = m[2 * N + i];
  float bx = 0.f, by = 0.f, bz = 0.f;
  if (mask & MM_DEMAG) { bx = bd[i]; by = bd[N + i]; bz = bd[2 * N + i]; }
  if ((mask & MM_EXCH) && (mask & MM_DMI_ON)) {
    if (lut->live[r] > 0.f) exch_dmi_cell(g, regions, lut, m, i, x, y, z, r, mx, my, mz, bx, by, bz);
  } else if (mask & MM_EXCH) {
    float ex = 0.f, ey = 0.f, ez = 0.f;
    auto nb = [&](long long j, float w) {
      float a = w * __ldg(&lut->exch[tri_index(r, regions[j])]);
      ex += a * (m[j] - mx); ey += a * (m[N + j] - my); ez += a * (m[2 * N + j] - mz);
    };
    if (g.Nx > 1) {
      if (x + 1 < g.Nx) nb(i + 1, g.inv_dx2); else if (g.pbc[0]) nb(i + 1 - g.Nx, g.inv_dx2);
      if (x > 0) nb(i - 1, g.inv_dx2); else if (g.pbc[0]) nb(i - 1 + g.Nx, g.inv_dx2);
    }
    if (g.Ny > 1) {
      const long long s = g.Nx;
      if (y + 1 < g.Ny) nb(i + s, g.inv_dy2); else if (g.pbc[1]) nb(i + s - s * g.Ny, g.inv_dy2);
      if (y > 0) nb(i - s, g.inv_dy2); else if (g.pbc[1]) nb(i - s + s * g.Ny, g.inv_dy2);
    }
    if (g.Nz > 1) {
      const long long s = (long long)g.Nx * g.Ny;
      if (z + 1 < g.Nz) nb(i + s, g.inv_dz2); else if (g.pbc[2]) nb(i + s - s * g.Nz, g.inv_dz2);
      if (z > 0) nb(i - s, g.inv_dz2); else if (g.pbc[2]) nb(i - s + s * g.Nz, g.inv_dz2);
    }
    bx += ex; by += ey; bz += ez;
  }
  if (mask & MM_ANIS) {
    if (lut->has_uniaxial) {
      float ux = lut->u[0][r], uy = lut->u[1][r], uz = lut->u[2][r];
      float um = ux * mx + uy * my + uz * mz;
      float s = lut->ku1[r] * um + lut->ku2[r] * um * um * um;
      bx += s * ux; by += s * uy; bz += s * uz;
    }
    if (lut->has_cubic) {
      float c1x = lut->c1[0][r], c1y = lut->c1[1][r], c1z = lut->c1[2][r];
      float c2x = lut->c2[0][r], c2y = lut->c2[1][r], c2z = lut->c2[2][r];
      float c3x = lut->c3[0][r], c3y = lut->c3[1][r], c3z = lut->c3[2][r];
      float a1 = c1x * mx + c1y * my + c1z * mz, a2 = c2x * mx + c2y * my + c2z * mz, a3 = c3x * mx + c3y * my + c3z * mz;
      float q1 = a1 * a1, q2 = a2 * a2, q3 = a3 * a3;
      float k1 = lut->kc1[r], k2 = lut->kc2[r], k3 = lut->kc3[r];
      float f1 = (k1 * (q2 + q3) + k2 * (q2 * q3) + k3 * (q2 * q2 + q3 * q3) * q1) * a1;
      float f2 = (k1 * (q1 + q3) + k2 * (q1 * q3) + k3 * (q1 * q1 + q3 * q3) * q2) * a2;
      float f3 = (k1 * (q1 + q2) + k2 * (q1 * q2) + k3 * (q1 * q1 + q2 * q2) * q3) * a3;
      bx += f1 * c1x + f2 * c2x + f3 * c3x;
      by += f1 * c1y + f2 * c2y + f3 * c3y;
      bz += f1 * c1z + f2 * c2z + f3 * c3z;
    }
  }
  if (mask & MM_ZEEMAN) { bx += lut->bext[0]; by += lut->bext[1]; bz += lut->bext[2]; }
  if (mask & MM_THERMAL) {     // Eq. 24: one eta per cell, component and step
    const float amp = lut->therm[r] * st->therm_scale;
    const unsigned long long idx = (unsigned long long)(st->steps + st->rejected) * (unsigned long long)N + (unsigned long long)i;
    bx += amp * mm_eta(st->seed, 0, idx); by += amp * mm_eta(st->seed, 1, idx); bz += amp * mm_eta(st->seed, 2, idx);
  }
  if (out_torque) {
    const float al = lut->alpha[r];
    const float pre = -lut->live[r] / (1.f + al * al);
    float tx = my * bz - mz * by, ty = mz * bx - mx * bz, tz = mx * by - my * bx;   // m x B
    float dx = my * tz - mz * ty, dy = mz * tx - mx * tz, dz = mx * ty - my * tx;   // m x (m x B)
    const float pr = out_torque == 1 ? 1.f : 0.f;      // out_torque == 2: precession term off (relax, L388)
      bx = pre * (pr * tx + al * dx); by = pre * (pr * ty + al * dy); bz = pre * (pr * tz + al * dz);
  }
  dst[i] = bx; dst[N + i] = by; dst[2 * N + i] = bz;
}

struct StageCoef { float a[6]; int n; };   // a_ij of one tableau row, n = number of slopes it combines
struct ErrCoef { float e[7]; };            // b(high) - b(low) of the embedded pair

// Same computation, four consecutive x cells per thread (Nx % 4 == 0): 16-byte loads of m, its y/z
// neighbour rows, B_demag and the region bytes; only the two x-edge neighbours are scalar loads.
// UNIFORM = one region: no region gathers, the exchange coefficient is a constant.
// THERMAL = add the fluctuating field of the current step (instantiated apart: it costs registers).
// FUSE = 1: the torque just formed is slope k_i; the kernel also forms the NEXT stage input
//          y_{i+1} = normalise(m0 + h gamma (sum_{j<i} a_j k_j + a_i k_i)) (sc = that tableau row, the last
//          coefficient belongs to k_i) into role ynext - a different buffer than the one the exchange
//          stencil is reading. Saves re-reading k_i and one launch per stage.
// FUSE = 2: last stage of a step: the error norm max || sum_j e_j k_j || (L372) is reduced here.
// grid = (Nx/4 / blockDim.x, Ny, Nz)
// DMI = a Dzyaloshinskii-Moriya strength is set: the exchange part runs cell by cell through exch_dmi_cell
//       (boundary conditions, virtual neighbours); instantiated apart, the hot path does not pay for it.
template <bool UNIFORM, bool THERMAL, int FUSE, bool DMI = false>
__global__ void __launch_bounds__(128) k_local4(Geometry g, const uint8_t* __restrict__ regions, const Luts* __restrict__ lut,
                                                DevState* st, int m_role, int bd_role, int dst_role, unsigned mask,
                                                int out_torque, StageCoef sc, ErrCoef ec, int ynext_role) {
  if (st->skip) return;
  const int x4 = blockIdx.x * blockDim.x + threadIdx.x;
  if (x4 * 4 >= g.Nx) return;
  const int x = x4 * 4, y = blockIdx.y, z = blockIdx.z;
  const long long N = g.N;
  const long long row = ((long long)z * g.Ny + y) * g.Nx;
  const long long i = row + x;
  const float* __restrict__ m = st->ptr[m_role];
  const float* __restrict__ bd = st->ptr[bd_role];
  float* __restrict__ dst = st->ptr[dst_role];
  float mc[3][4], b[3][4];
  int r[4] = {0, 0, 0, 0};
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float4 q = *reinterpret_cast<const float4*>(m + c * N + i);
    mc[c][0] = q.x; mc[c][1] = q.y; mc[c][2] = q.z; mc[c][3] = q.w;
    if (mask & MM_DEMAG) {
      const float4 d = *reinterpret_cast<const float4*>(bd + c * N + i);
      b[c][0] = d.x; b[c][1] = d.y; b[c][2] = d.z; b[c][3] = d.w;
    } else {
      b[c][0] = b[c][1] = b[c][2] = b[c][3] = 0.f;
    }
  }
  if (!UNIFORM) {
    const uchar4 q = *reinterpret_cast<const uchar4*>(regions + i);
    r[0] = q.x; r[1] = q.y; r[2] = q.z; r[3] = q.w;
  }
  if (DMI && (mask & MM_EXCH)) {
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      const int rl = UNIFORM ? 0 : r[l];
      if (lut->live[rl] > 0.f)
        exch_dmi_cell(g, regions, lut, m, i + l, x + l, y, z, rl, mc[0][l], mc[1][l], mc[2][l], b[0][l], b[1][l], b[2][l]);
    }
  } else if (mask & MM_EXCH) {
    const float a0 = lut->exch[0];
    // a whole neighbour row segment (y or z direction): j = index of its first cell
    auto nb_row = [&](long long j, float w) {
      int rn[4] = {0, 0, 0, 0};
      if (!UNIFORM) {
        const uchar4 q = *reinterpret_cast<const uchar4*>(regions + j);
        rn[0] = q.x; rn[1] = q.y; rn[2] = q.z; rn[3] = q.w;
      }
      float a[4];
#pragma unroll
      for (int l = 0; l < 4; ++l) a[l] = w * (UNIFORM ? a0 : __ldg(&lut->exch[tri_index(r[l], rn[l])]));
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float4 q = *reinterpret_cast<const float4*>(m + c * N + j);
        b[c][0] += a[0] * (q.x - mc[c][0]); b[c][1] += a[1] * (q.y - mc[c][1]);
        b[c][2] += a[2] * (q.z - mc[c][2]); b[c][3] += a[3] * (q.w - mc[c][3]);
      }
    };
    // one neighbour cell j of lane l
    auto nb_one = [&](int l, long long j, float w) {
      const float a = w * (UNIFORM ? a0 : __ldg(&lut->exch[tri_index(r[l], regions[j])]));
#pragma unroll
      for (int c = 0; c < 3; ++c) b[c][l] += a * (m[c * N + j] - mc[c][l]);
    };
    if (g.Nx > 1) {
      const float w = g.inv_dx2;
      // interior x neighbours come from the registers
#pragma unroll
      for (int l = 0; l < 3; ++l) {
        const float a = w * (UNIFORM ? a0 : __ldg(&lut->exch[tri_index(r[l], r[l + 1])]));
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float d = mc[c][l + 1] - mc[c][l];
          b[c][l] += a * d; b[c][l + 1] -= a * d;
        }
      }
      if (x > 0) nb_one(0, i - 1, w); else if (g.pbc[0]) nb_one(0, row + g.Nx - 1, w);
      if (x + 4 < g.Nx) nb_one(3, i + 4, w); else if (g.pbc[0]) nb_one(3, row, w);
    }
    if (g.Ny > 1) {
      const long long s = g.Nx;
      if (y + 1 < g.Ny) nb_row(i + s, g.inv_dy2); else if (g.pbc[1]) nb_row(i + s - s * g.Ny, g.inv_dy2);
      if (y > 0) nb_row(i - s, g.inv_dy2); else if (g.pbc[1]) nb_row(i - s + s * g.Ny, g.inv_dy2);
    }
    if (g.Nz > 1) {
      const long long s = (long long)g.Nx * g.Ny;
      if (z + 1 < g.Nz) nb_row(i + s, g.inv_dz2); else if (g.pbc[2]) nb_row(i + s - s * g.Nz, g.inv_dz2);
      if (z > 0) nb_row(i - s, g.inv_dz2); else if (g.pbc[2]) nb_row(i - s + s * g.Nz, g.inv_dz2);
    }
  }
  const bool uni = (mask & MM_ANIS) && lut->has_uniaxial, cub = (mask & MM_ANIS) && lut->has_cubic;
#pragma unroll
  for (int l = 0; l < 4; ++l) {
    const int rr = r[l];
    const float mx = mc[0][l], my = mc[1][l], mz = mc[2][l];
    float bx = b[0][l], by = b[1][l], bz = b[2][l];
    if (uni) {
      float ux = lut->u[0][rr], uy = lut->u[1][rr], uz = lut->u[2][rr];
      float um = ux * mx + uy * my + uz * mz;
      float sc = lut->ku1[rr] * um + lut->ku2[rr] * um * um * um;
      bx += sc * ux; by += sc * uy; bz += sc * uz;
    }
    if (cub) {
      float c1x = lut->c1[0][rr], c1y = lut->c1[1][rr], c1z = lut->c1[2][rr];
      float c2x = lut->c2[0][rr], c2y = lut->c2[1][rr], c2z = lut->c2[2][rr];
      float c3x = lut->c3[0][rr], c3y = lut->c3[1][rr], c3z = lut->c3[2][rr];
      float a1 = c1x * mx + c1y * my + c1z * mz, a2 = c2x * mx + c2y * my + c2z * mz, a3 = c3x * mx + c3y * my + c3z * mz;
      float q1 = a1 * a1, q2 = a2 * a2, q3 = a3 * a3;
      float k1 = lut->kc1[rr], k2 = lut->kc2[rr], k3 = lut->kc3[rr];
      float f1 = (k1 * (q2 + q3) + k2 * (q2 * q3) + k3 * (q2 * q2 + q3 * q3) * q1) * a1;
      float f2 = (k1 * (q1 + q3) + k2 * (q1 * q3) + k3 * (q1 * q1 + q3 * q3) * q2) * a2;
      float f3 = (k1 * (q1 + q2) + k2 * (q1 * q2) + k3 * (q1 * q1 + q2 * q2) * q3) * a3;
      bx += f1 * c1x + f2 * c2x + f3 * c3x;
      by += f1 * c1y + f2 * c2y + f3 * c3y;
      bz += f1 * c1z + f2 * c2z + f3 * c3z;
    }
    if (mask & MM_ZEEMAN) { bx += lut->bext[0]; by += lut->bext[1]; bz += lut->bext[2]; }
    if (THERMAL) {             // Eq. 24: one eta per cell, component and step
      const float amp = lut->therm[rr] * st->therm_scale;
      const unsigned long long idx = (unsigned long long)(st->steps + st->rejected) * (unsigned long long)N + (unsigned long long)(i + l);
      bx += amp * mm_eta(st->seed, 0, idx); by += amp * mm_eta(st->seed, 1, idx); bz += amp * mm_eta(st->seed, 2, idx);
    }
    if (out_torque) {
      const float al = lut->alpha[rr];
      const float pre = -lut->live[rr] / (1.f + al * al);
      float tx = my * bz - mz * by, ty = mz * bx - mx * bz, tz = mx * by - my * bx;   // m x B
      float dx = my * tz - mz * ty, dy = mz * tx - mx * tz, dz = mx * ty - my * tx;   // m x (m x B)
      const float pr = out_torque == 1 ? 1.f : 0.f;      // out_torque == 2: precession term off (relax, L388)
      bx = pre * (pr * tx + al * dx); by = pre * (pr * ty + al * dy); bz = pre * (pr * tz + al * dz);
    }
    b[0][l] = bx; b[1][l] = by; b[2][l] = bz;
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) *reinterpret_cast<float4*>(dst + c * N + i) = make_float4(b[c][0], b[c][1], b[c][2], b[c][3]);
  if (FUSE == 1) {
    float sv[3][4];
    float al = 0.f;
#pragma unroll
    for (int j = 0; j < 6; ++j) al = (j == sc.n - 1) ? sc.a[j] : al;      // coefficient of the slope just formed
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int l = 0; l < 4; ++l) sv[c][l] = al * b[c][l];
#pragma unroll
    for (int j = 0; j < 5; ++j) {
      if (j < sc.n - 1 && sc.a[j] != 0.f) {
        const float* __restrict__ k = st->ptr[R_K0 + j];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float4 q = *reinterpret_cast<const float4*>(k + c * N + i);
          sv[c][0] += sc.a[j] * q.x; sv[c][1] += sc.a[j] * q.y; sv[c][2] += sc.a[j] * q.z; sv[c][3] += sc.a[j] * q.w;
        }
      }
    }
    const float* __restrict__ m0 = st->ptr[R_M];
    float* __restrict__ yn = st->ptr[ynext_role];
    const float hg = st->hg;
    float y[3][4];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float4 q = *reinterpret_cast<const float4*>(m0 + c * N + i);
      y[c][0] = q.x + hg * sv[c][0]; y[c][1] = q.y + hg * sv[c][1]; y[c][2] = q.z + hg * sv[c][2]; y[c][3] = q.w + hg * sv[c][3];
    }
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      const float n2 = y[0][l] * y[0][l] + y[1][l] * y[1][l] + y[2][l] * y[2][l];
      const float inv = n2 > 0.f ? rsqrtf(n2) : 0.f;
      y[0][l] *= inv; y[1][l] *= inv; y[2][l] *= inv;
    }
#pragma unroll
    for (int c = 0; c < 3; ++c) *reinterpret_cast<float4*>(yn + c * N + i) = make_float4(y[c][0], y[c][1], y[c][2], y[c][3]);
  }
  if (FUSE == 2) {
    float sv[3][4];
    const int last = dst_role - R_K0;
    float el = 0.f;
#pragma unroll
    for (int j = 0; j < 7; ++j) el = (j == last) ? ec.e[j] : el;          // weight of the slope just formed
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int l = 0; l < 4; ++l) sv[c][l] = el * b[c][l];
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      if (j < last && ec.e[j] != 0.f) {
        const float* __restrict__ k = st->ptr[R_K0 + j];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float4 q = *reinterpret_cast<const float4*>(k + c * N + i);
          sv[c][0] += ec.e[j] * q.x; sv[c][1] += ec.e[j] * q.y; sv[c][2] += ec.e[j] * q.z; sv[c][3] += ec.e[j] * q.w;
        }
      }
    }
    float best = 0.f;
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      const float n = sqrtf(sv[0][l] * sv[0][l] + sv[1][l] * sv[1][l] + sv[2][l] * sv[2][l]);
      best = (n > best || n != n) ? n : best;          // NaN propagates
    }
    // warp maximum over the lanes that are here (a ragged last block has partial warps); non-negative
    // floats order like their bit patterns, NaN is mapped above +inf
    const unsigned act = __activemask();
    const unsigned bits = __reduce_max_sync(act, (best != best) ? 0x7fc00000u : __float_as_uint(best));
    if ((int)(threadIdx.x & 31) == __ffs(act) - 1) atomicMax(&st->err_bits, bits);
  }
}

// Dormand-Prince stage input y_i = normalise(m0 + h sum_j a_ij k_j) (L365; every stage input is
// renormalised, reading #9). k_j are torques over gamma [T], hg = gamma * h.

__global__ void k_stage(long long N, DevState* st, StageCoef sc, int dst_role) {
  if (st->skip) return;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const float* __restrict__ m = st->ptr[R_M];
  const float hg = st->hg;
  float sx = 0.f, sy = 0.f, sz = 0.f;
#pragma unroll
  for (int j = 0; j < 6; ++j) {
    if (j < sc.n && sc.a[j] != 0.f) {
      const float* __restrict__ k = st->ptr[R_K0 + j];
      sx += sc.a[j] * k[i]; sy += sc.a[j] * k[N + i]; sz += sc.a[j] * k[2 * N + i];
    }
  }
  float yx = m[i] + hg * sx, yy = m[N + i] + hg * sy, yz = m[2 * N + i] + hg * sz;
  float n2 = yx * yx + yy * yy + yz * yz;
  float inv = n2 > 0.f ? rsqrtf(n2) : 0.f;
  float* __restrict__ dst = st->ptr[dst_role];
  dst[i] = yx * inv; dst[N + i] = yy * inv; dst[2 * N + i] = yz * inv;
}

// the same with four cells per thread and 16-byte accesses (N a multiple of 4: every component starts 16-byte aligned);
// per cell the arithmetic and its order are those of k_stage
__global__ void __launch_bounds__(256) k_stage4(long long N, DevState* st, StageCoef sc, int dst_role) {
  if (st->skip) return;
  const long long i = 4 * ((long long)blockIdx.x * blockDim.x + threadIdx.x);
  if (i >= N) return;
  const float* __restrict__ m = st->ptr[R_M];
  const float hg = st->hg;
  float s[3][4];
#pragma unroll
  for (int c = 0; c < 3; ++c)
#pragma unroll
    for (int l = 0; l < 4; ++l) s[c][l] = 0.f;
#pragma unroll
  for (int j = 0; j < 6; ++j) {
    if (j < sc.n && sc.a[j] != 0.f) {
      const float* __restrict__ k = st->ptr[R_K0 + j];
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float4 q = *reinterpret_cast<const float4*>(k + c * N + i);
        s[c][0] += sc.a[j] * q.x; s[c][1] += sc.a[j] * q.y; s[c][2] += sc.a[j] * q.z; s[c][3] += sc.a[j] * q.w;
      }
    }
  }
  float y[3][4];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float4 q = *reinterpret_cast<const float4*>(m + c * N + i);
    y[c][0] = q.x + hg * s[c][0]; y[c][1] = q.y + hg * s[c][1]; y[c][2] = q.z + hg * s[c][2]; y[c][3] = q.w + hg * s[c][3];
  }
#pragma unroll
  for (int l = 0; l < 4; ++l) {
    const float n2 = y[0][l] * y[0][l] + y[1][l] * y[1][l] + y[2][l] * y[2][l];
    const float inv = n2 > 0.f ? rsqrtf(n2) : 0.f;
    y[0][l] *= inv; y[1][l] *= inv; y[2][l] *= inv;
  }
  float* __restrict__ dst = st->ptr[dst_role];
#pragma unroll
  for (int c = 0; c < 3; ++c) *reinterpret_cast<float4*>(dst + c * N + i) = make_float4(y[c][0], y[c][1], y[c][2], y[c][3]);
}

// eps / h = max_cells || sum_j e_j k_j ||_2   (L372; Euclidean norm, reading #8)

__global__ void k_error(long long N, DevState* st, ErrCoef ec) {
  if (st->skip) return;
  float best = 0.f;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    float sx = 0.f, sy = 0.f, sz = 0.f;
#pragma unroll
    for (int j = 0; j < 7; ++j) {
      if (ec.e[j] != 0.f) {
        const float* __restrict__ k = st->ptr[R_K0 + j];
        sx += ec.e[j] * k[i]; sy += ec.e[j] * k[N + i]; sz += ec.e[j] * k[2 * N + i];
      }
    }
    float n = sqrtf(sx * sx + sy * sy + sz * sz);
    best = (n > best || n != n) ? n : best;          // NaN propagates
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    float other = __shfl_xor_sync(0xffffffffu, best, o);
    best = (other > best || other != other) ? other : best;
  }
  if ((threadIdx.x & 31) == 0) {
    unsigned bits = (best != best) ? 0x7fc00000u : __float_as_uint(best);   // NaN sorts above +inf
    atomicMax(&st->err_bits, bits);
  }
}

// Step-size control on the device (single thread each).
// begin: choose the step h of this attempt; in run mode clip it to land exactly on t_end
// (reading #10) or mark the run as finished (skip = 1: the rest of the step is a no-op).
__global__ void k_ctrl_begin(DevState* st) {
  if (st->status != MM_OK) { st->skip = 1; return; }
  double h = st->fix_dt > 0 ? st->fix_dt : st->dt;
  st->clipped = 0;
  if (st->run_mode) {
    double remaining = st->t_end - st->t;
    if (!(remaining > 1e-12 * fmax(st->run_duration, 1e-30))) { st->skip = 1; return; }
    if (h >= remaining) { st->keep_dt = h; h = remaining; st->clipped = 1; }
  }
  st->skip = 0;
  st->h = h;
  st->hg = (float)(st->gamma * h);
  st->therm_scale = (float)sqrt(st->temperature / h);
  st->err_bits = 0u;
}

// end: eps = h * max|...|; accept iff fixed step or eps <= MaxErr; on accept swap the roles
// m <-> y7 and k1 <-> k7 (FSAL); dt <- dt * headroom * clamp((MaxErr/eps)^(1/5), 0.5, 2) (L372-L374,
// DESIGN.md readings #7-#9).
__global__ void k_ctrl_end(DevState* st) {
  if (st->skip) return;
  const float emax = __uint_as_float(st->err_bits);
  const double h = st->h;
  const double err = (double)emax * st->gamma * h;
  st->last_err = (float)err;
  st->evals += st->nevals;
  if (!(err == err) || isinf(err)) { st->status = MM_ENAN; st->last_accepted = 0; st->skip = 1; return; }
  const bool fixed = st->fix_dt > 0;
  const bool accept = fixed || err <= st->max_err;
  st->last_accepted = accept ? 1 : 0;
  if (accept) {
    float* p = st->ptr[R_M]; st->ptr[R_M] = st->ptr[R_MNEW]; st->ptr[R_MNEW] = p;
    const int last = R_K0 + st->nstage - 1;          // FSAL: the last stage slope is the next first one
    p = st->ptr[R_K0]; st->ptr[R_K0] = st->ptr[last]; st->ptr[last] = p;
    st->t = st->clipped ? st->t_end : st->t + h;
    st->steps += 1;
  } else {
    st->rejected += 1;
  }
  if (!fixed) {
    if (accept && st->clipped) {
      st->dt = st->keep_dt;
    } else {
      double fac = (err == 0.0) ? 2.0 : fmin(2.0, fmax(0.5, pow(st->max_err / err, st->expo)));
      double dt = h * st->headroom * fac;
      dt = fmin(st->dt_max, fmax(st->dt_min, dt));
      if (!accept && h <= st->dt_min) { st->status = MM_EDT; st->skip = 1; }
      st->dt = dt;
    }
  }
}

// effective region map of a box with a geometry (mm_set_geometry): cells outside the shape take the reserved
// vacuum index (its look-up-table entries are zero: no B_sat, no exchange)
#define MM_VACUUM_REGION (MM_MAX_REGIONS - 1)
__global__ void k_apply_geometry(long long N, const uint8_t* __restrict__ user, const uint8_t* __restrict__ inside,
                                 uint8_t* __restrict__ out) {
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x)
    out[i] = inside[i] ? user[i] : (uint8_t)MM_VACUUM_REGION;
}

// largest region id of the map (validated against nregions without copying the map to the host)
__global__ void k_max_region(long long N, const uint8_t* __restrict__ regions, unsigned* __restrict__ out) {
  unsigned best = 0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x)
    best = max(best, (unsigned)regions[i]);
  best = __reduce_max_sync(0xffffffffu, best);
  if ((threadIdx.x & 31) == 0 && best > 0) atomicMax(out, best);
}

// diagnostics (mm_b_eff, mm_torque, mm_energy, mm_max_torque) evaluate fields whatever the state of the last
// step: a failed step (MM_ENAN / MM_EDT) leaves skip = 1 until the error is cleared
__global__ void k_clear_skip(DevState* st) { st->skip = 0; }

// |m| = 1 on entry (L85); vacuum cells (Msat = 0) and zero vectors stay 0
__global__ void k_normalise(long long N, float* __restrict__ m, const uint8_t* __restrict__ regions,
                            const Luts* __restrict__ lut) {
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  float x = m[i], y = m[N + i], z = m[2 * N + i];
  float n2 = x * x + y * y + z * z;
  float inv = (n2 > 0.f ? rsqrtf(n2) : 0.f) * lut->live[regions[i]];
  m[i] = x * inv; m[N + i] = y * inv; m[2 * N + i] = z * inv;
}

// Deterministic grid-wide fp64 sum of NV values per thread: warp shuffles, the warps of a block in index order,
// one partial per block, and the block that finishes last (ticket counter) adds the partials in block order and
// resets the ticket. The result does not depend on scheduling, so the same state always gives the same bits
// (batched and one-at-a-time runs compare energies with ==). part: gridDim.x * NV doubles; ticket: zero on entry.
template <int NV>
__device__ __forceinline__ void grid_sum_ordered(double* v, double* __restrict__ part, unsigned* __restrict__ ticket,
                                                 double* __restrict__ out) {
  __shared__ double wsum[32][NV];
  __shared__ bool last;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
  for (int c = 0; c < NV; ++c) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    if (lane == 0) wsum[w][c] = v[c];
  }
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int c = 0; c < NV; ++c) {
      double a = 0.0;
      for (int i = 0; i < nw; ++i) a += wsum[i][c];
      part[(size_t)blockIdx.x * NV + c] = a;
    }
    __threadfence();
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  if (threadIdx.x < NV) {
    double a = 0.0;
    for (unsigned b = 0; b < gridDim.x; ++b) a += __ldcg(&part[(size_t)b * NV + threadIdx.x]);
    out[threadIdx.x] = a;
  }
  if (threadIdx.x == 0) *ticket = 0u;
}

// plain mean of m (fp64 accumulation, fixed summation order)
__global__ void k_sum3(long long N, const float* __restrict__ m, double* __restrict__ part, unsigned* __restrict__ ticket,
                       double* __restrict__ out) {
  double s[3] = {0.0, 0.0, 0.0};
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    s[0] += m[i]; s[1] += m[N + i]; s[2] += m[2 * N + i];
  }
  grid_sum_ordered<3>(s, part, ticket, out);
}

// Energy of the selected terms, joules / cell volume summed over cells (fp64 accumulation):
//   E/V = - sum_cells M . [ 1/2 B_demag (Eq. 4) + 1/2 B_exch (Eq. 8) + 1/2 B_anis(Ku1) + 1/4 B_anis(Ku2) (Eq. 20)
//                           + 1/4 B(Kc1) + 1/6 B(Kc2) + 1/8 B(Kc3) (Eq. 23) + B_ext ],   M = Msat m.
// B_demag of m must already be in role bd_role. Fixed summation order (grid_sum_ordered).
__global__ void k_energy(Geometry g, const uint8_t* __restrict__ regions, const Luts* __restrict__ lut, DevState* st,
                         int m_role, int bd_role, unsigned mask, double* __restrict__ part, unsigned* __restrict__ ticket,
                         double* __restrict__ out) {
  const float* __restrict__ m = st->ptr[m_role];
  const float* __restrict__ bd = st->ptr[bd_role];
  const long long N = g.N;
  double acc = 0.0;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    const int x = (int)(i % g.Nx);
    const long long t = i / g.Nx;
    const int y = (int)(t % g.Ny), z = (int)(t / g.Ny);
    const int r = regions[i];
    const float mx = m[i], my = m[N + i], mz = m[2 * N + i];
    float e = 0.f;                                      // sum of weight * m . B  [T]
    if (mask & MM_DEMAG) e += 0.5f * (mx * bd[i] + my * bd[N + i] + mz * bd[2 * N + i]);
    if ((mask & MM_EXCH) && (mask & MM_DMI_ON)) {       // Eq. 8 + Eq. 17: -1/2 M . (B_exch + B_DM)
      float ex = 0.f, ey = 0.f, ez = 0.f;
      if (lut->live[r] > 0.f) exch_dmi_cell(g, regions, lut, m, i, x, y, z, r, mx, my, mz, ex, ey, ez);
      e += 0.5f * (mx * ex + my * ey + mz * ez);
    } else if (mask & MM_EXCH) {
      float ex = 0.f, ey = 0.f, ez = 0.f;
      auto nb = [&](long long j, float w) {
        float a = w * __ldg(&lut->exch[tri_index(r, regions[j])]);
        ex += a * (m[j] - mx); ey += a * (m[N + j] - my); ez += a * (m[2 * N + j] - mz);
      };
      if (g.Nx > 1) {
        if (x + 1 < g.Nx) nb(i + 1, g.inv_dx2); else if (g.pbc[0]) nb(i + 1 - g.Nx, g.inv_dx2);
        if (x > 0) nb(i - 1, g.inv_dx2); else if (g.pbc[0]) nb(i - 1 + g.Nx, g.inv_dx2);
      }
      if (g.Ny > 1) {
        const long long s = g.Nx;
        if (y + 1 < g.Ny) nb(i + s, g.inv_dy2); else if (g.pbc[1]) nb(i + s - s * g.Ny, g.inv_dy2);
        if (y > 0) nb(i - s, g.inv_dy2); else if (g.pbc[1]) nb(i - s + s * g.Ny, g.inv_dy2);
      }
      if (g.Nz > 1) {
        const long long s = (long long)g.Nx * g.Ny;
        if (z + 1 < g.Nz) nb(i + s, g.inv_dz2); else if (g.pbc[2]) nb(i + s - s * g.Nz, g.inv_dz2);
        if (z > 0) nb(i - s, g.inv_dz2); else if (g.pbc[2]) nb(i - s + s * g.Nz, g.inv_dz2);
      }
      e += 0.5f * (mx * ex + my * ey + mz * ez);
    }
    if (mask & MM_ANIS) {
      if (lut->has_uniaxial) {
        const float um = lut->u[0][r] * mx + lut->u[1][r] * my + lut->u[2][r] * mz, u2 = um * um;
        e += 0.5f * lut->ku1[r] * u2 + 0.25f * lut->ku2[r] * u2 * u2;
      }
      if (lut->has_cubic) {
        const float a1 = lut->c1[0][r] * mx + lut->c1[1][r] * my + lut->c1[2][r] * mz;
        const float a2 = lut->c2[0][r] * mx + lut->c2[1][r] * my + lut->c2[2][r] * mz;
        const float a3 = lut->c3[0][r] * mx + lut->c3[1][r] * my + lut->c3[2][r] * mz;
        const float q1 = a1 * a1, q2 = a2 * a2, q3 = a3 * a3;
        e += 0.25f * lut->kc1[r] * 2.f * (q1 * q2 + q1 * q3 + q2 * q3) + (1.f / 6.f) * lut->kc2[r] * 3.f * q1 * q2 * q3 +
             0.125f * lut->kc3[r] * 2.f * (q1 * q1 * q2 * q2 + q1 * q1 * q3 * q3 + q2 * q2 * q3 * q3);
      }
    }
    if (mask & MM_ZEEMAN) e += mx * lut->bext[0] + my * lut->bext[1] + mz * lut->bext[2];
    acc -= (double)lut->Bsat[r] * (double)e;           // times mu0 Msat; divided by mu0 on the host
  }
  grid_sum_ordered<1>(&acc, part, ticket, out);
}

// max over cells of the Euclidean norm of a 3N vector field (float bits; non-negative floats order as uints)
__global__ void k_maxnorm(long long N, const float* __restrict__ v, unsigned* __restrict__ out) {
  float best = 0.f;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    const float x = v[i], y = v[N + i], z = v[2 * N + i];
    const float n = sqrtf(x * x + y * y + z * z);
    best = (n > best || n != n) ? n : best;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const float other = __shfl_xor_sync(0xffffffffu, best, o);
    best = (other > best || other != other) ? other : best;
  }
  if ((threadIdx.x & 31) == 0) atomicMax(out, (best != best) ? 0x7fc00000u : __float_as_uint(best));
}

// Slonczewski spin-transfer torque (Eq. 28-30) over gamma_LL [T], added to the torque in role
// tq_role for the magnetisation in role m_role (a kernel of its own: the hot path does not pay for it):
//   tau_SL = beta (eps - alpha eps')/(1+alpha^2) m x (m_P x m) - beta (eps' - alpha eps)/(1+alpha^2) m x m_P,
//   beta = j_z hbar / (Msat e d) = pref / Bsat,  eps = P L^2 / ((L^2+1) + (L^2-1) m.m_P).
struct SttArgs { float pref, pol, lam2, eps_prime, mp[3]; };   // pref = j_z hbar mu0 / (e d)  [T^2]

__global__ void k_add_stt(long long N, const uint8_t* __restrict__ regions, const Luts* __restrict__ lut, DevState* st,
                          int m_role, int tq_role, SttArgs p) {
  if (st->skip) return;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= N) return;
  const float* __restrict__ m = st->ptr[m_role];
  float* __restrict__ tq = st->ptr[tq_role];
  const int r = regions[i];
  const float bs = lut->Bsat[r];
  if (!(bs > 0.f)) return;
  const float al = lut->alpha[r], beta = p.pref / bs, den = 1.f / (1.f + al * al);
  const float mx = m[i], my = m[N + i], mz = m[2 * N + i];
  const float px = p.mp[0], py = p.mp[1], pz = p.mp[2];
  const float c = mx * px + my * py + mz * pz;
  const float eps = p.pol * p.lam2 / ((p.lam2 + 1.f) + (p.lam2 - 1.f) * c);
  const float a = beta * (eps - al * p.eps_prime) * den, b = -beta * (p.eps_prime - al * eps) * den;
  // m x (m_P x m) = m_P - (m.m_P) m for |m| = 1, written out as the double cross product
  const float qx = py * mz - pz * my, qy = pz * mx - px * mz, qz = px * my - py * mx;      // m_P x m
  const float dx = my * qz - mz * qy, dy = mz * qx - mx * qz, dz = mx * qy - my * qx;      // m x (m_P x m)
  const float ex = my * pz - mz * py, ey = mz * px - mx * pz, ez = mx * py - my * px;      // m x m_P
  tq[i] += a * dx + b * ex; tq[N + i] += a * dy + b * ey; tq[2 * N + i] += a * dz + b * ez;
}

// Zhang-Li spin-transfer torque (Eq. 26; #19) over gamma_LL [T], added to the torque in
// role tq_role:  1/(1+alpha^2) [ (1 + xi alpha) m x (m x D) + (xi - alpha) m x D ],  D = (u . grad) m,
// u = mu_B mu0 j / (2 e gamma_LL Bsat (1 + xi^2)); central differences, a missing neighbour at an open
// boundary is the cell's own m (L196), periodic axes wrap.
struct ZlArgs { float c[3]; float xi; };     // c[a] = mu_B mu0 j_a / (2 e gamma (1 + xi^2)) / (2 d_a)  [T^2]

__global__ void k_add_zl(Geometry g, const uint8_t* __restrict__ regions, const Luts* __restrict__ lut, DevState* st,
                         int m_role, int tq_role, ZlArgs p) {
  if (st->skip) return;
  const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= g.N) return;
  const long long N = g.N;
  const float* __restrict__ m = st->ptr[m_role];
  float* __restrict__ tq = st->ptr[tq_role];
  const int r = regions[i];
  const float bs = lut->Bsat[r];
  if (!(bs > 0.f)) return;
  const int x = (int)(i % g.Nx);
  const long long t = i / g.Nx;
  const int y = (int)(t % g.Ny), z = (int)(t / g.Ny);
  float dx = 0.f, dy = 0.f, dz = 0.f;
  auto diff = [&](long long up, long long dn, float c) {
    if (!(lut->Bsat[regions[up]] > 0.f)) up = i;       // a vacuum neighbour is a missing neighbour: own m (L196, L53)
    if (!(lut->Bsat[regions[dn]] > 0.f)) dn = i;
    dx += c * (m[up] - m[dn]); dy += c * (m[N + up] - m[N + dn]); dz += c * (m[2 * N + up] - m[2 * N + dn]);
  };
  if (g.Nx > 1 && p.c[0] != 0.f) {
    const long long up = x + 1 < g.Nx ? i + 1 : (g.pbc[0] ? i + 1 - g.Nx : i), dn = x > 0 ? i - 1 : (g.pbc[0] ? i - 1 + g.Nx : i);
    diff(up, dn, p.c[0] / bs);
  }
  if (g.Ny > 1 && p.c[1] != 0.f) {
    const long long s = g.Nx;
    const long long up = y + 1 < g.Ny ? i + s : (g.pbc[1] ? i + s - s * g.Ny : i), dn = y > 0 ? i - s : (g.pbc[1] ? i - s + s * g.Ny : i);
    diff(up, dn, p.c[1] / bs);
  }
  if (g.Nz > 1 && p.c[2] != 0.f) {
    const long long s = (long long)g.Nx * g.Ny;
    const long long up = z + 1 < g.Nz ? i + s : (g.pbc[2] ? i + s - s * g.Nz : i), dn = z > 0 ? i - s : (g.pbc[2] ? i - s + s * g.Nz : i);
    diff(up, dn, p.c[2] / bs);
  }
  const float al = lut->alpha[r], den = 1.f / (1.f + al * al);
  const float mx = m[i], my = m[N + i], mz = m[2 * N + i];
  const float ex = my * dz - mz * dy, ey = mz * dx - mx * dz, ez = mx * dy - my * dx;      // m x D
  const float fx = my * ez - mz * ey, fy = mz * ex - mx * ez, fz = mx * ey - my * ex;      // m x (m x D)
  const float a = (1.f + p.xi * al) * den, b = (p.xi - al) * den;
  tq[i] += a * fx + b * ex; tq[N + i] += a * fy + b * ey; tq[2 * N + i] += a * fz + b * ez;
}
