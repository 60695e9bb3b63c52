// Host loop of bemcub_solve (included by bemcub.cu): right-preconditioned restarted GMRES around
// the potential-only evaluation kernel.  SURVEY.md §8(f).2; PAPER.md L34 (the BEM system for the
// unknown charge densities), L200 (matrix elements computed on the fly, matrix not stored).
// Where the caller allows it and 8 n^2 bytes fit (bemcub_solve_storage; 180 GB of HBM hold n = 1.4e5),
// the matrix is filled once by the matrix-fill kernel and every mat-vec is an HBM-bound GEMV.
namespace {

constexpr int kGmresRestart = 30;

struct SolveWork {
  double* cen;    // [n][3] element centroids = field points of the mat-vec
  double* diag;   // [n]    A_ii
  double* basis;  // [restart + 1][n]
  double* w;      // [n]
  double* z;      // [n]
  double* coef;   // [3 * (restart + 2)]: first and second Gram-Schmidt pass, then |w|^2; also y of the update
  const double* matrix;  // [n][n] when the solve keeps it, else null
};

inline unsigned blocks_for(int64_t n) { return (unsigned)((n + 255) / 256); }

// out = A * x   (one adaptive potential-only evaluation at the centroids; the sort is reused)
int solve_matvec(bemcub_ctx* c, const bemcub_policy* pol, const SolveWork& k, const double* x, double* out, bool first) {
  if (k.matrix) return bemcub_matvec(c, k.matrix, c->n, x, out);
  return eval_common(c, x, BEMCUB_RULE_ADAPTIVE, pol, c->n, k.cen, out, nullptr, nullptr, BEMCUB_F64, !first);
}

// dev_out[v] = V[v] . w for v < nvec (deterministic tree reduction, one block per vector); stays on the device
int dots_dev(bemcub_ctx* c, int nvec, const double* basis, const double* w, double* dev_out) {
  const int64_t n = c->n;
  vec_dots_kernel<<<nvec, 1024, 0, c->stream>>>(n, basis, n, w, dev_out);
  c->stats.kernel_launches += 1;
  CUDA_TRY(cudaGetLastError());
  return BEMCUB_OK;
}

int to_host(bemcub_ctx* c, const double* dev, int count, double* host) {
  CUDA_TRY(cudaMemcpyAsync(host, dev, sizeof(double) * count, cudaMemcpyDeviceToHost, c->stream));
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  return BEMCUB_OK;
}

}  // namespace

extern "C" int bemcub_matvec(bemcub_ctx* c, const double* matrix, int64_t ld, const double* x, double* y) {
  if (!c) return BEMCUB_ERR_INVALID_ARG;
  if (!c->has_mesh) return BEMCUB_ERR_NO_ELEMENTS;
  const int64_t n = c->n;
  if (n == 0) return BEMCUB_OK;
  if (!matrix || !x || !y || ld < n || x == y) return BEMCUB_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  const int grid = (int)std::min<int64_t>(n, (int64_t)c->num_sms * kGemvCtasPerSm);
  gemv_rows_kernel<<<grid, kGemvThreads, 0, c->stream>>>(n, matrix, ld, x, y);
  count_launch(c);
  CUDA_TRY(cudaGetLastError());
  return BEMCUB_OK;
}

extern "C" int bemcub_solve_storage(bemcub_ctx* c, int64_t max_matrix_bytes) {
  if (!c || max_matrix_bytes < 0) return BEMCUB_ERR_INVALID_ARG;
  c->solve_matrix_limit = max_matrix_bytes;
  if (max_matrix_bytes == 0) {
    DeviceGuard g(c->device);
    cudaStreamSynchronize(c->stream);
    release(c->solve_matrix);
  }
  return BEMCUB_OK;
}

extern "C" int bemcub_solve(bemcub_ctx* c, const bemcub_policy* host_policy, const double* rhs, double* sigma, double rel_tol,
                            int max_matvecs, int* host_matvecs, double* host_rel_residual) {
  if (!c || !host_policy) return BEMCUB_ERR_INVALID_ARG;
  if (!c->has_mesh) return BEMCUB_ERR_NO_ELEMENTS;
  if (!(rel_tol > 0.0) || max_matvecs < 1) return BEMCUB_ERR_INVALID_ARG;
  if (host_matvecs) *host_matvecs = 0;
  if (host_rel_residual) *host_rel_residual = 0.0;
  const int64_t n = c->n;
  if (n == 0) return BEMCUB_OK;
  if (!rhs || !sigma) return BEMCUB_ERR_INVALID_ARG;
  PolicyDev pd;
  int rc = build_policy(host_policy, &pd);
  if (rc) return rc;
  DeviceGuard g(c->device);
  const int M = kGmresRestart;
  if ((rc = ensure(c->solve_buf[0], (size_t)n * 24)) || (rc = ensure(c->solve_buf[1], (size_t)n * 8)) ||
      (rc = ensure(c->solve_buf[2], (size_t)(M + 1) * n * 8)) || (rc = ensure(c->solve_buf[3], (size_t)n * 8)) ||
      (rc = ensure(c->solve_buf[4], (size_t)n * 8)) || (rc = ensure(c->solve_buf[5], (size_t)3 * (M + 2) * 8)))
    return rc;
  SolveWork k;
  k.cen = (double*)c->solve_buf[0].ptr;
  k.diag = (double*)c->solve_buf[1].ptr;
  k.basis = (double*)c->solve_buf[2].ptr;
  k.w = (double*)c->solve_buf[3].ptr;
  k.z = (double*)c->solve_buf[4].ptr;
  k.coef = (double*)c->solve_buf[5].ptr;
  k.matrix = nullptr;
  if (n <= ((int64_t)1 << 30) && (int64_t)sizeof(double) * n * n <= c->solve_matrix_limit) {
    if ((rc = ensure(c->solve_matrix, sizeof(double) * (size_t)n * (size_t)n))) return rc;
    if ((rc = bemcub_assemble_rows(c, host_policy, 0, n, (double*)c->solve_matrix.ptr, n))) return rc;
    k.matrix = (const double*)c->solve_matrix.ptr;
  }
  CUDA_TRY(cudaMemcpy2DAsync(k.cen, 24, c->cenL.ptr, 32, 24, (size_t)n, cudaMemcpyDeviceToDevice, c->stream));
  self_term_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, (const uint8_t*)c->type.ptr, (const double*)c->verts.ptr,
                                                        (const double4*)c->cenL.ptr, coulomb_k(), k.diag);
  c->stats.kernel_launches += 1;
  CUDA_TRY(cudaGetLastError());

  double hb = 0.0;
  if ((rc = dots_dev(c, 1, rhs, rhs, k.coef)) || (rc = to_host(c, k.coef, 1, &hb))) return rc;
  const double bnorm = std::sqrt(hb);
  if (bnorm == 0.0) {  // zero potential everywhere: zero charge
    CUDA_TRY(cudaMemsetAsync(sigma, 0, (size_t)n * 8, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
    return BEMCUB_OK;
  }
  int matvecs = 0;
  bool first = true;
  double relres = 1.0;
  bool converged = false;
  double H[kGmresRestart + 1][kGmresRestart], cs[kGmresRestart], sn[kGmresRestart], gv[kGmresRestart + 1];
  double hbuf[3 * (kGmresRestart + 2)];
  const int stride = M + 2;  // coef = [pass 1 | pass 2 | norm]

  // Every cycle starts with the true residual of the current iterate, so the residual reported at the
  // end is always that of the sigma returned; the Arnoldi loop leaves one mat-vec of the budget for it.
  while (matvecs < max_matvecs) {
    // true residual r = b - A x, V_0 = r / |r|
    if ((rc = solve_matvec(c, host_policy, k, sigma, k.w, first))) return rc;
    first = false;
    ++matvecs;
    vec_sub_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, rhs, k.w, k.w);
    double rr = 0.0;
    if ((rc = dots_dev(c, 1, k.w, k.w, k.coef)) || (rc = to_host(c, k.coef, 1, &rr))) return rc;
    c->stats.kernel_launches += 1;
    const double beta = std::sqrt(rr);
    relres = beta / bnorm;
    if (relres <= rel_tol) {
      converged = true;
      break;
    }
    if (matvecs >= max_matvecs) break;
    vec_scale_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, 1.0 / beta, k.w, nullptr, k.basis);
    gv[0] = beta;
    int j = 0;
    for (; j < M && matvecs < max_matvecs - 1; ++j) {
      // w = A M^-1 V_j
      vec_scale_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, 1.0, k.basis + (int64_t)j * n, k.diag, k.z);
      if ((rc = solve_matvec(c, host_policy, k, k.z, k.w, false))) return rc;
      ++matvecs;
      // classical Gram-Schmidt, twice; coefficients, norm and the new basis vector all stay on the
      // device - ONE copy to the host per step, for the Hessenberg column and the stopping test
      if ((rc = dots_dev(c, j + 1, k.basis, k.w, k.coef))) return rc;
      vec_combine_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, j + 1, k.basis, n, k.coef, -1.0, k.w);
      if ((rc = dots_dev(c, j + 1, k.basis, k.w, k.coef + stride))) return rc;
      vec_combine_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, j + 1, k.basis, n, k.coef + stride, -1.0, k.w);
      if ((rc = dots_dev(c, 1, k.w, k.w, k.coef + 2 * stride))) return rc;
      vec_normalise_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, k.w, k.coef + 2 * stride, k.basis + (int64_t)(j + 1) * n);
      c->stats.kernel_launches += 4;
      if ((rc = to_host(c, k.coef, 2 * stride + 1, hbuf))) return rc;
      const double hnext = std::sqrt(hbuf[2 * stride]);
      for (int i = 0; i <= j; ++i) H[i][j] = hbuf[i] + hbuf[stride + i];
      // Givens rotations of the new Hessenberg column
      for (int i = 0; i < j; ++i) {
        const double t = cs[i] * H[i][j] + sn[i] * H[i + 1][j];
        H[i + 1][j] = -sn[i] * H[i][j] + cs[i] * H[i + 1][j];
        H[i][j] = t;
      }
      const double den = std::hypot(H[j][j], hnext);
      cs[j] = den > 0.0 ? H[j][j] / den : 1.0;
      sn[j] = den > 0.0 ? hnext / den : 0.0;
      H[j][j] = den;
      gv[j + 1] = -sn[j] * gv[j];
      gv[j] = cs[j] * gv[j];
      const double est = std::fabs(gv[j + 1]) / bnorm;
      if (est <= rel_tol || hnext == 0.0) {
        ++j;
        break;
      }
    }
    // y = H^-1 g (upper triangular), x += M^-1 sum y_i V_i
    double y[kGmresRestart];
    for (int i = j - 1; i >= 0; --i) {
      double t = gv[i];
      for (int l = i + 1; l < j; ++l) t -= H[i][l] * y[l];
      y[i] = t / H[i][i];
    }
    if (j > 0) {
      CUDA_TRY(cudaMemcpyAsync(k.coef, y, sizeof(double) * j, cudaMemcpyHostToDevice, c->stream));
      CUDA_TRY(cudaMemsetAsync(k.z, 0, (size_t)n * 8, c->stream));
      vec_combine_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, j, k.basis, n, k.coef, 1.0, k.z);
      vec_add_scaled_kernel<<<blocks_for(n), 256, 0, c->stream>>>(n, k.z, k.diag, sigma);
      c->stats.kernel_launches += 2;
      CUDA_TRY(cudaStreamSynchronize(c->stream));  // y lives on the host stack
    }
    CUDA_TRY(cudaGetLastError());
  }
  CUDA_TRY(cudaStreamSynchronize(c->stream));
  if (host_matvecs) *host_matvecs = matvecs;
  if (host_rel_residual) *host_rel_residual = relres;
  return converged ? BEMCUB_OK : BEMCUB_ERR_NOT_CONVERGED;
}
