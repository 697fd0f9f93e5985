// setup.cu - demagnetising-kernel set-up (see demag_setup.cuh)
#include <algorithm>
#include "internal.cuh"
#include "demag_setup.cuh"

// ---- demag kernel set-up (fp64 on the device)
// layouts: bit 0 = the generic K[comp][kz][ky][kx], bit 1 = the fast 2D layout Kt (only if the box has that path)
int mm_build_kernel_spectrum(mm_sim* s, int layouts) {
  const Geometry& g = s->g;
  setup::TensorGrid tg;
  tg.N[0] = g.Nx; tg.N[1] = g.Ny; tg.N[2] = g.Nz;
  tg.P[0] = g.Px; tg.P[1] = g.Py; tg.P[2] = g.Pz;
  for (int a = 0; a < 3; ++a) {
    tg.rep[a] = s->rep[a];
    tg.d[a] = s->cell[a];
    tg.E[a] = s->rep[a] > 0 ? tg.N[a] / 2 + 1 : tg.N[a];
  }
  const long long noct = (long long)tg.E[0] * tg.E[1] * tg.E[2];
  const long long nfull = (long long)g.Px * g.Py * g.Pz;
  const int ncomp = (g.Nz == 1 && s->rep[2] == 0) ? 4 : 6;
  const long long nk = (long long)g.Cx * g.Hy * g.Hz;
  const bool want_k = (layouts & 1) != 0, want_kt = (layouts & 2) != 0 && s->fast2d;
  if (want_k) {
    s->K = (float*)mm_dev_alloc(s, sizeof(float) * nk * ncomp);
    if (!s->K) return mm_fail(s, MM_ENOMEM, "kernel spectrum");
  }
  const int fNy = g.Py / 2;      // transform length along y of the fast path
  const long long nkt = (long long)g.Cx * (fNy + 1);
  if (want_kt) {
    s->Kt = (float*)mm_dev_alloc(s, sizeof(float) * nkt * 4);
    if (!s->Kt) return mm_fail(s, MM_ENOMEM, "kernel spectrum (fast layout)");
  }
  double* oct = (double*)mm_dev_alloc(s, sizeof(double) * noct * 6);
  double2* bufA = (double2*)mm_dev_alloc(s, sizeof(double2) * nfull);
  double2* bufB = (double2*)mm_dev_alloc(s, sizeof(double2) * nfull);
  double* maxim = (double*)mm_dev_alloc(s, sizeof(double));
  if (!oct || !bufA || !bufB || !maxim) return mm_fail(s, MM_ENOMEM, "kernel set-up scratch");
  CUDA_TRY(s, cudaMemsetAsync(maxim, 0, sizeof(double), s->stream));
  setup::k_tensor_octant<<<blocks_for(noct, 128), 128, 0, s->stream>>>(tg, oct);
  s->launches++;
  CUDA_TRY(s, cudaGetLastError());
  const double scale = 1.0 / ((double)g.Px * g.Py * g.Pz);
  for (int comp = 0; comp < ncomp; ++comp) {
    setup::k_expand<<<blocks_for(nfull, 256), 256, 0, s->stream>>>(tg, oct, comp, bufA);
    s->launches++;
    double2* src = bufA;
    double2* dst = bufB;
    const AxisPlan* plans[3] = {&s->px, &s->py, &s->pz};
    long long stride = 1;
    for (int a = 0; a < 3; ++a) {
      const AxisPlan& pl = *plans[a];
      int Ns = 1;
      for (int p = 0; p < pl.npass; ++p) {
        int R = pl.radix[p];
        long long total = nfull / R;
        setup::k_fft_pass_f64<<<blocks_for(total, 256), 256, 0, s->stream>>>(src, dst, total, pl.P, R, Ns, stride);
        s->launches++;
        Ns *= R;
        std::swap(src, dst);
      }
      stride *= pl.P;
    }
    if (want_k) {
      setup::k_pack_spectrum<<<blocks_for(nk, 256), 256, 0, s->stream>>>(tg, src, s->K + (size_t)comp * nk, g.Cx, g.Hy, g.Hz,
                                                                         scale, maxim);
      s->launches++;
    }
    if (want_kt) {
      setup::k_pack_spectrum_2dfast<<<blocks_for(nkt, 256), 256, 0, s->stream>>>(tg, src, s->Kt + (size_t)comp * nkt, g.Cx,
                                                                                 fNy, scale);
      s->launches++;
    }
    CUDA_TRY(s, cudaGetLastError());
  }
  double him = 0.0;
  CUDA_TRY(s, cudaMemcpyAsync(&him, maxim, sizeof(double), cudaMemcpyDeviceToHost, s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  mm_dev_free(s, oct); mm_dev_free(s, bufA); mm_dev_free(s, bufB); mm_dev_free(s, maxim);
  if (him > 1e-6) return mm_fail(s, MM_ECUDA, "kernel spectrum is not real: max |Im| = " + std::to_string(him));
  return MM_OK;
}

