// Model construction: hyper-parameter checks, blob parsing, weight upload, tensor-track tables.
// (SURVEY.md §8(b) boundary and blob layout; PAPER.md:222 for what the MLPs are.)
#include <nvtx3/nvToolsExt.h>
#include <cmath>
#include <cstring>

#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "internal.h"

static thread_local std::string g_err;

void al_set_error(const allegro_model* m, const std::string& msg) {
  g_err = msg;
  if (m) const_cast<allegro_model*>(m)->err = msg;
}

extern "C" const char* allegro_last_error(const allegro_model* m) { return m ? m->err.c_str() : g_err.c_str(); }

int al_alloc(allegro_model* m, void** p, size_t bytes) {
  *p = nullptr;
  if (bytes == 0) bytes = 16;
  if (m && m->alloc_fn) {
    *p = m->alloc_fn(bytes, m->alloc_user);
    if (!*p) { al_set_error(m, "allocator hook returned NULL"); return ALLEGRO_ERR_CUDA; }
    return ALLEGRO_OK;
  }
  AL_CUDA(m, cudaMalloc(p, bytes));
  return ALLEGRO_OK;
}

void al_free(allegro_model* m, void* p) {
  if (!p) return;
  if (m && m->free_fn) m->free_fn(p, m->alloc_user);
  else cudaFree(p);
}

int al_reserve(allegro_model* m, DevBuf& b, size_t bytes) {
  if (b.bytes >= bytes && b.p) return ALLEGRO_OK;
  if (b.p) { cudaStreamSynchronize(m->stream); al_free(m, b.p); b.p = nullptr; b.bytes = 0; }
  if (m) m->alloc_gen++;
  size_t want = bytes + bytes / 20 + 256;   // +5 % head-room (avoid allocator churn)
  AL_CHECK(al_alloc(m, &b.p, want));
  b.bytes = want;
  return ALLEGRO_OK;
}

void al_release(allegro_model* m, DevBuf& b) {
  if (b.p) al_free(m, b.p);
  b.p = nullptr; b.bytes = 0;
}

static int check_hp(const allegro_hparams* hp) {
  if (!hp) { al_set_error(nullptr, "hparams is NULL"); return ALLEGRO_ERR_BAD_ARG; }
  auto bad = [&](const char* s) { al_set_error(nullptr, std::string("bad hparams: ") + s); return ALLEGRO_ERR_BAD_HPARAMS; };
  if (hp->n_species < 1 || hp->n_species > 64) return bad("n_species");
  if (hp->l_max < 0 || hp->l_max > 3) return bad("l_max must be in [0,3]");
  if (hp->n_layers < 1 || hp->n_layers > AL_MAX_LAYERS) return bad("n_layers");
  if (hp->n_tensor < 1 || hp->n_tensor % 4) return bad("n_tensor must be a positive multiple of 4");
  if (hp->n_bessel < 1 || hp->n_bessel > 16) return bad("n_bessel");
  if (hp->poly_p < 2 || hp->poly_p > 32) return bad("poly_p");
  if (!(hp->r_cut > 0)) return bad("r_cut");
  if (hp->n_twobody < 1 || hp->n_twobody > 8 || hp->n_latent < 1 || hp->n_latent > 8 || hp->n_edge < 0 || hp->n_edge > 8)
    return bad("MLP depth");
  for (int k = 0; k < hp->n_twobody; ++k) if (hp->twobody_dims[k] < 4 || hp->twobody_dims[k] % 4) return bad("twobody_dims (multiples of 4)");
  for (int k = 0; k < hp->n_latent; ++k) if (hp->latent_dims[k] < 4 || hp->latent_dims[k] % 4) return bad("latent_dims (multiples of 4)");
  for (int k = 0; k < hp->n_edge; ++k) if (hp->edge_dims[k] < 1) return bad("edge_dims");
  if (hp->latent_dims[hp->n_latent - 1] != hp->twobody_dims[hp->n_twobody - 1]) return bad("last latent width must equal d");
  if (!(hp->avg_num_neighbors > 0)) return bad("avg_num_neighbors");
  if (hp->precision < 0 || hp->precision > 4) return bad("precision");
  if (hp->precision == 2 || hp->precision == 4) {
    // 16-bit operand MLPs (tcgen05 kind::f16): TMA rows of 16-bit tensors need 16-byte strides, the K-concatenated x-bar GEMM
    // needs a first latent width that is a multiple of the 64-element k-block, and the fused last-latent epilogue d % 32 == 0
    if (hp->n_twobody < 2) return bad("16-bit operand modes need at least two two-body layers");
    for (int k = 0; k < hp->n_twobody; ++k) if (hp->twobody_dims[k] % 8) return bad("16-bit operand modes: twobody_dims multiples of 8");
    for (int k = 0; k < hp->n_latent; ++k) if (hp->latent_dims[k] % 8) return bad("16-bit operand modes: latent_dims multiples of 8");
    if (hp->latent_dims[0] % 64) return bad("16-bit operand modes: first latent width a multiple of 64");
    if (hp->twobody_dims[hp->n_twobody - 1] % 32 || hp->n_tensor % 32) return bad("16-bit operand modes: d and n_tensor multiples of 32");
  }
  return ALLEGRO_OK;
}

static void n_paths_of(const allegro_hparams* hp, std::vector<int>& np) {
  std::vector<std::vector<Irrep>> S;
  std::vector<std::vector<TPLayerHost::Path>> paths;
  al_enumerate(hp->l_max, hp->n_layers, S, paths);
  np.clear();
  for (auto& p : paths) np.push_back((int)p.size());
}

static size_t blob_floats(const allegro_hparams* hp) {
  std::vector<int> np;
  n_paths_of(hp, np);
  size_t S = hp->n_species, NB = hp->n_bessel, d = hp->twobody_dims[hp->n_twobody - 1], n = hp->n_tensor;
  size_t nA = n * (hp->l_max + 1), tot = 0, fi = 2 * S + NB;
  for (int k = 0; k < hp->n_twobody; ++k) { tot += fi * hp->twobody_dims[k]; fi = hp->twobody_dims[k]; }
  tot += d * nA;
  for (int L = 0; L < hp->n_layers; ++L) {
    tot += d * nA + np[L];
    fi = d + n;
    for (int k = 0; k < hp->n_latent; ++k) { tot += fi * hp->latent_dims[k]; fi = hp->latent_dims[k]; }
  }
  fi = d;
  for (int k = 0; k < hp->n_edge; ++k) { tot += fi * hp->edge_dims[k]; fi = hp->edge_dims[k]; }
  tot += fi;
  return tot;
}

extern "C" int allegro_blob_size(const allegro_hparams* hp, size_t* bytes) {
  AL_CHECK(check_hp(hp));
  if (!bytes) return ALLEGRO_ERR_BAD_ARG;
  size_t b = blob_floats(hp) * 4;
  b += (8 - b % 8) % 8;
  *bytes = b + 16 * (size_t)hp->n_species;
  return ALLEGRO_OK;
}

extern "C" int allegro_path_info(const allegro_hparams* hp, int32_t layer, int32_t* n_paths, int32_t* fan, int32_t* dims) {
  AL_CHECK(check_hp(hp));
  if (layer < 1 || layer > hp->n_layers) { al_set_error(nullptr, "layer out of range"); return ALLEGRO_ERR_BAD_ARG; }
  allegro_model tmp;
  tmp.lmax = hp->l_max; tmp.NL = hp->n_layers; tmp.Denv = (hp->l_max + 1) * (hp->l_max + 1);
  AL_CHECK(al_build_tp_tables(&tmp, {}));
  const TPLayerHost& t = tmp.tp_host[layer - 1];
  if (n_paths) *n_paths = (int32_t)t.paths.size();
  if (fan) for (size_t k = 0; k < t.fan.size(); ++k) fan[k] = t.fan[k];
  if (dims) { dims[0] = t.Din; dims[1] = t.Dout; }
  return ALLEGRO_OK;
}

template <typename T>
static int upload(allegro_model* m, T** dst, const std::vector<T>& h) {
  void* p;   // weights and tables: plain cudaMalloc (created before an allocator hook can be set)
  AL_CUDA(m, cudaMalloc(&p, h.size() * sizeof(T) + 16));
  m->owned.push_back(p);
  if (!h.empty()) AL_CUDA(m, cudaMemcpy(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
  *dst = (T*)p;
  return ALLEGRO_OK;
}

void al_gemm_tc_free(allegro_model* m);   // gemm_tc.cu

static int upload_dense(allegro_model* m, Dense& D, const std::vector<float>& W, int fi, int fo) {
  D.fi = fi; D.fo = fo;
  std::vector<float> Wt((size_t)fi * fo);
  for (int i = 0; i < fi; ++i)
    for (int o = 0; o < fo; ++o) Wt[(size_t)o * fi + i] = W[(size_t)i * fo + o];
  AL_CHECK(upload(m, &D.W, W));
  AL_CHECK(upload(m, &D.Wt, Wt));
  if (m->hfmt >= 0) {
    auto conv = [&](const std::vector<float>& x) {
      std::vector<uint16_t> h(x.size());
      for (size_t k = 0; k < x.size(); ++k) {
        if (m->hfmt == 0) { __half v = __float2half_rn(x[k]); memcpy(&h[k], &v, 2); }
        else { __nv_bfloat16 v = __float2bfloat16_rn(x[k]); memcpy(&h[k], &v, 2); }
      }
      return h;
    };
    uint16_t* p16 = nullptr;
    AL_CHECK(upload(m, &p16, conv(W))); D.W16 = p16;
    AL_CHECK(upload(m, &p16, conv(Wt))); D.Wt16 = p16;
  }
  if (m->hp.precision == 0) {
    auto split = [](const std::vector<float>& x, std::vector<float>& hi, std::vector<float>& lo) {
      hi.resize(x.size()); lo.resize(x.size());
      auto rn = [](float v) { uint32_t b; memcpy(&b, &v, 4); b = (b + 0x1000u) & 0xFFFFE000u; float r; memcpy(&r, &b, 4); return r; };
      for (size_t k = 0; k < x.size(); ++k) {
        hi[k] = rn(x[k]);
        lo[k] = rn(x[k] - hi[k]);
      }
    };
    std::vector<float> hi, lo;
    split(W, hi, lo);
    AL_CHECK(upload(m, &D.W_hi, hi)); AL_CHECK(upload(m, &D.W_lo, lo));
    split(Wt, hi, lo);
    AL_CHECK(upload(m, &D.Wt_hi, hi)); AL_CHECK(upload(m, &D.Wt_lo, lo));
  }
  return ALLEGRO_OK;
}

extern "C" int allegro_create(const allegro_hparams* hp, const void* blob, size_t blob_bytes, allegro_model** out) {
  if (!out || !blob) { al_set_error(nullptr, "NULL argument"); return ALLEGRO_ERR_BAD_ARG; }
  *out = nullptr;
  AL_CHECK(check_hp(hp));
  size_t want;
  AL_CHECK(allegro_blob_size(hp, &want));
  if (want != blob_bytes) {
    al_set_error(nullptr, "blob size mismatch: expected " + std::to_string(want) + " bytes, got " + std::to_string(blob_bytes));
    return ALLEGRO_ERR_BLOB_SIZE;
  }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    al_set_error(nullptr, "no CUDA device: libb200allegro has no CPU fallback");
    return ALLEGRO_ERR_CUDA;
  }
  allegro_model* m = new allegro_model();
  m->hp = *hp;
  m->hfmt = (hp->precision == 2) ? 1 : (hp->precision == 4) ? 0 : -1;
  m->S = hp->n_species; m->NB = hp->n_bessel; m->d = hp->twobody_dims[hp->n_twobody - 1];
  m->n = hp->n_tensor; m->lmax = hp->l_max; m->NL = hp->n_layers;
  m->Denv = (m->lmax + 1) * (m->lmax + 1); m->nA = m->n * (m->lmax + 1); m->ldY = (m->Denv + 3) & ~3;
  int dev = 0; cudaGetDevice(&dev);
  m->device = dev;
  cudaDeviceGetAttribute(&m->sm_count, cudaDevAttrMultiProcessorCount, dev);
  m->c_env = (float)(1.0 / std::sqrt(hp->avg_num_neighbors));
  for (int L = 0; L < m->NL; ++L) {
    double a = hp->resid_alpha[L];
    m->c_old[L] = (float)(1.0 / std::sqrt(1.0 + a * a));
    m->c_new[L] = (float)(a / std::sqrt(1.0 + a * a));
  }
  const float* f = (const float*)blob;
  size_t o = 0;
  auto take = [&](size_t cnt) { std::vector<float> v(f + o, f + o + cnt); o += cnt; return v; };
  int rc = ALLEGRO_OK;
  auto fail = [&](int r) { allegro_destroy(m); return r; };
  // two-body
  int fi = 2 * m->S + m->NB;
  m->twobody.resize(hp->n_twobody);
  for (int k = 0; k < hp->n_twobody; ++k) {
    int fo = hp->twobody_dims[k];
    if ((rc = upload_dense(m, m->twobody[k], take((size_t)fi * fo), fi, fo))) return fail(rc);
    fi = fo;
  }
  // embeddings: permute columns (n, l) -> (l, n)
  auto permute = [&](const std::vector<float>& A) {
    std::vector<float> P(A.size());
    int nl = m->lmax + 1;
    for (int r = 0; r < m->d; ++r)
      for (int nn = 0; nn < m->n; ++nn)
        for (int l = 0; l < nl; ++l) P[(size_t)r * m->nA + l * m->n + nn] = A[(size_t)r * m->nA + nn * nl + l];
    return P;
  };
  std::vector<float> A0 = permute(take((size_t)m->d * m->nA));
  std::vector<std::vector<float>> alphas(m->NL);
  std::vector<int> npaths;
  n_paths_of(hp, npaths);
  m->emb.resize(m->NL + 1);
  m->latent.resize(m->NL);
  m->xcat.resize(m->NL); m->sbar.resize(m->NL);
  std::vector<float> A01_keep;
  for (int L = 1; L <= m->NL; ++L) {
    std::vector<float> AL = permute(take((size_t)m->d * m->nA));
    alphas[L - 1] = take(npaths[L - 1]);
    if (L == 1) {
      std::vector<float> A01((size_t)m->d * 2 * m->nA);
      for (int r = 0; r < m->d; ++r) {
        memcpy(&A01[(size_t)r * 2 * m->nA], &A0[(size_t)r * m->nA], m->nA * 4);
        memcpy(&A01[(size_t)r * 2 * m->nA + m->nA], &AL[(size_t)r * m->nA], m->nA * 4);
      }
      if ((rc = upload_dense(m, m->emb01, A01, m->d, 2 * m->nA))) return fail(rc);
      A01_keep = A01;
    } else {
      if ((rc = upload_dense(m, m->emb[L - 1], AL, m->d, m->nA))) return fail(rc);
    }
    fi = m->d + m->n;
    m->latent[L - 1].resize(hp->n_latent);
    for (int k = 0; k < hp->n_latent; ++k) {
      int fo = hp->latent_dims[k];
      std::vector<float> Wk = take((size_t)fi * fo);
      if ((rc = upload_dense(m, m->latent[L - 1][k], Wk, fi, fo))) return fail(rc);
      if (k == 0) {
        // K-concatenated weights of the x-bar GEMM and the s-bar rows (see internal.h)
        const std::vector<float>& Ae = (L == 1) ? A01_keep : AL;
        const int Kx = (L == 1) ? 2 * m->nA : m->nA, h = fo, d = m->d;
        std::vector<float> cat((size_t)d * (h + Kx)), sb((size_t)m->n * h);
        for (int r = 0; r < d; ++r) {
          memcpy(&cat[(size_t)r * (h + Kx)], &Wk[(size_t)r * h], (size_t)h * 4);
          memcpy(&cat[(size_t)r * (h + Kx) + h], &Ae[(size_t)r * Kx], (size_t)Kx * 4);
        }
        memcpy(sb.data(), &Wk[(size_t)d * h], (size_t)m->n * h * 4);
        if ((rc = upload_dense(m, m->xcat[L - 1], cat, d, h + Kx))) return fail(rc);
        if ((rc = upload_dense(m, m->sbar[L - 1], sb, m->n, h))) return fail(rc);
      }
      fi = fo;
    }
  }
  // edge MLP has no nonlinearity: collapse to one d-vector in fp64
  {
    std::vector<double> v;
    fi = m->d;
    std::vector<std::vector<float>> Ws; std::vector<int> fos;
    for (int k = 0; k <= hp->n_edge; ++k) {
      int fo = (k < hp->n_edge) ? hp->edge_dims[k] : 1;
      Ws.push_back(take((size_t)fi * fo)); fos.push_back(fo); fi = fo;
    }
    // v = W_0 W_1 ... W_last  ([d] x 1), evaluated right to left
    v.assign(1, 1.0);
    for (int k = (int)Ws.size() - 1; k >= 0; --k) {
      int fo = fos[k]; int fin = (int)(Ws[k].size() / fo);
      std::vector<double> nv(fin, 0.0);
      for (int i = 0; i < fin; ++i) { double s = 0; for (int c = 0; c < fo; ++c) s += (double)Ws[k][(size_t)i * fo + c] * v[c]; nv[i] = s; }
      v = nv;
    }
    std::vector<float> vf(v.begin(), v.end());
    if ((rc = upload(m, &m->w_eff_d, v))) return fail(rc);
    if ((rc = upload(m, &m->w_eff_f, vf))) return fail(rc);
  }
  o += (2 - o % 2) % 2;
  const double* tail = (const double*)(f + o);
  m->sigma_h.assign(tail, tail + m->S);
  m->mu_h.assign(tail + m->S, tail + 2 * m->S);
  if ((rc = upload(m, &m->sigma, m->sigma_h))) return fail(rc);
  if ((rc = upload(m, &m->mu, m->mu_h))) return fail(rc);
  // tensor-track tables
  if ((rc = al_build_tp_tables(m, alphas))) return fail(rc);
  m->tp.resize(m->NL);
  for (int L = 0; L < m->NL; ++L) {
    TPLayerHost& h = m->tp_host[L]; TPLayerDev& t = m->tp[L];
    t.Din = h.Din; t.Dout = h.Dout; t.Denv = h.Denv; t.npairs = h.npairs; t.nnz = h.nnz;
    if ((rc = upload(m, &t.pair_a, h.pair_a)) || (rc = upload(m, &t.pair_c, h.pair_c)) ||
        (rc = upload(m, &t.pair_ptr, h.pair_ptr)) || (rc = upload(m, &t.ent_b, h.ent_b)) ||
        (rc = upload(m, &t.ent_val, h.ent_val)) || (rc = upload(m, &t.ent_idx, h.ent_idx)) || (rc = upload(m, &t.c_ptr, h.c_ptr)) ||
        (rc = upload(m, &t.c_a, h.c_a)) || (rc = upload(m, &t.c_p, h.c_p)) || (rc = upload(m, &t.a_ptr, h.a_ptr)) ||
        (rc = upload(m, &t.a_c, h.a_c)) || (rc = upload(m, &t.a_p, h.a_p)) || (rc = upload(m, &t.b_ptr, h.b_ptr)) ||
        (rc = upload(m, &t.b_p, h.b_p)) || (rc = upload(m, &t.b_val, h.b_val)) ||
        (rc = upload(m, &t.ce_pack, h.ce_pack)) || (rc = upload(m, &t.cent_ptr, h.cent_ptr)) || (rc = upload(m, &t.ce_val, h.ce_val)) ||
        (rc = upload(m, &t.ae_pack, h.ae_pack)) || (rc = upload(m, &t.aent_ptr, h.aent_ptr)) || (rc = upload(m, &t.ae_val, h.ae_val)) ||
        (rc = upload(m, &t.dp_ptr, h.dp_ptr)) || (rc = upload(m, &t.dp_b, h.dp_b)) || (rc = upload(m, &t.dp_val, h.dp_val)))
      return fail(rc);
  }
  std::vector<int> env_l;
  for (int l = 0; l <= m->lmax; ++l) for (int k = 0; k < 2 * l + 1; ++k) env_l.push_back(l);
  if ((rc = upload(m, &m->d_env_l, env_l)) || (rc = upload(m, &m->d_v0_l, m->v0_l)) || (rc = upload(m, &m->d_v0_y, m->v0_y)))
    return fail(rc);
  *out = m;
  return ALLEGRO_OK;
}

extern "C" int allegro_destroy(allegro_model* m) {
  if (!m) return ALLEGRO_OK;
  cudaDeviceSynchronize();
  al_work_free(m);
  al_gemm_tc_free(m);
  for (auto& r : m->prof_recs) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
  for (auto e : m->prof_pool) cudaEventDestroy(e);
  for (void* p : m->owned) cudaFree(p);
  if (m->sg.exec) cudaGraphExecDestroy(m->sg.exec);
  if (m->sg.cap) cudaStreamDestroy(m->sg.cap);
  delete m;
  return ALLEGRO_OK;
}

extern "C" int allegro_set_stream(allegro_model* m, void* s) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  m->stream = (cudaStream_t)s;   // (part of the step-graph key itself)
  return ALLEGRO_OK;
}

extern "C" int allegro_set_allocator(allegro_model* m, allegro_alloc_fn a, allegro_free_fn f, void* user) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  if (m->work) { al_set_error(m, "allocator must be set before the first compute call"); return ALLEGRO_ERR_BAD_ARG; }
  m->alloc_fn = a; m->free_fn = f; m->alloc_user = user;
  m->config_gen++;
  return ALLEGRO_OK;
}

extern "C" int allegro_set_pair_cutoffs(allegro_model* m, const double* rc_pair) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  AL_CUDA(m, cudaStreamSynchronize(m->stream));
  m->config_gen++;
  if (!rc_pair) { m->d_rc_pair = nullptr; return ALLEGRO_OK; }   // (the device array stays owned by the model)
  const int S = m->S;
  for (int k = 0; k < S * S; ++k)
    if (!(rc_pair[k] > 0) || rc_pair[k] > m->hp.r_cut) {
      al_set_error(m, "pair cutoffs must be in (0, r_cut]");
      return ALLEGRO_ERR_BAD_HPARAMS;
    }
  std::vector<double> h(rc_pair, rc_pair + (size_t)S * S);
  double* d = nullptr;
  AL_CHECK(upload(m, &d, h));
  m->d_rc_pair = d;
  return ALLEGRO_OK;
}

extern "C" int allegro_set_bessel_frequencies(allegro_model* m, const double* freq) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  AL_CUDA(m, cudaStreamSynchronize(m->stream));
  m->config_gen++;
  if (!freq) { m->d_bfreq = nullptr; return ALLEGRO_OK; }
  const size_t cnt = (size_t)m->S * m->S * m->NB;
  for (size_t k = 0; k < cnt; ++k)
    if (!(freq[k] > 0) || !std::isfinite(freq[k])) { al_set_error(m, "Bessel frequencies must be finite and > 0"); return ALLEGRO_ERR_BAD_HPARAMS; }
  std::vector<double> h(freq, freq + cnt);
  double* d = nullptr;
  AL_CHECK(upload(m, &d, h));
  m->d_bfreq = d;
  return ALLEGRO_OK;
}

extern "C" int allegro_set_zbl(allegro_model* m, const double* atomic_numbers) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  AL_CUDA(m, cudaStreamSynchronize(m->stream));
  m->config_gen++;
  if (!atomic_numbers) { m->d_zbl_Z = nullptr; return ALLEGRO_OK; }
  for (int k = 0; k < m->S; ++k)
    if (!(atomic_numbers[k] > 0) || !std::isfinite(atomic_numbers[k])) { al_set_error(m, "atomic numbers must be > 0"); return ALLEGRO_ERR_BAD_HPARAMS; }
  std::vector<double> h(atomic_numbers, atomic_numbers + m->S);
  double* d = nullptr;
  AL_CHECK(upload(m, &d, h));
  m->d_zbl_Z = d;
  return ALLEGRO_OK;
}

extern "C" int allegro_set_tensor_track(allegro_model* m, int32_t mode) {
  if (!m || (mode != 0 && mode != 1)) return ALLEGRO_ERR_BAD_ARG;
  if (m->work_sized) { al_set_error(m, "the tensor-track mode must be set before the first compute call"); return ALLEGRO_ERR_BAD_ARG; }
  m->tt_mode = mode;
  m->config_gen++;
  return ALLEGRO_OK;
}

extern "C" int allegro_set_debug(allegro_model* m, int on) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  m->debug_keep = on != 0;
  m->config_gen++;
  return ALLEGRO_OK;
}

extern "C" int allegro_set_chunk_edges(allegro_model* m, int64_t e) {
  if (!m || e < 1024) return ALLEGRO_ERR_BAD_ARG;
  m->chunk_edges = e;
  m->config_gen++;
  return ALLEGRO_OK;
}

extern "C" int allegro_launch_count(const allegro_model* m, int64_t* l) {
  if (!m || !l) return ALLEGRO_ERR_BAD_ARG;
  *l = m->launches;
  return ALLEGRO_OK;
}

// ---- per-kernel-group event timing ---------------------------------------------------------------------
static cudaEvent_t prof_event(allegro_model* m) {
  if (!m->prof_pool.empty()) { cudaEvent_t e = m->prof_pool.back(); m->prof_pool.pop_back(); return e; }
  cudaEvent_t e; cudaEventCreate(&e); return e;
}
static const char* kProfNames[PC_COUNT] = {"gemm", "tp_fwd", "tp_bwd", "geom", "twobody0", "energy", "bwd_elem", "edge_bwd",
                                           "neighbors", "nve"};

ProfScope::ProfScope(allegro_model* m_, int cat_) : m(m_), cat(cat_) {
  if (m && m->nvtx) { nvtxRangePushA(kProfNames[cat]); range = true; }   // e.g. ncu --nvtx --nvtx-include "gemm/"
  if (m && m->prof) { a = prof_event(m); cudaEventRecord(a, m->stream); }
}
ProfScope::~ProfScope() {
  if (a) { cudaEvent_t b = prof_event(m); cudaEventRecord(b, m->stream); m->prof_recs.push_back({cat, a, b}); }
  if (range) nvtxRangePop();
}

extern "C" int allegro_set_gemm_pairs(allegro_model* m, int32_t pairs) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  m->gemm_cta_pairs = pairs != 0;
  m->config_gen++;          // a captured step graph holds the old launch shapes
  return ALLEGRO_OK;
}

extern "C" int allegro_profile_enable(allegro_model* m, int32_t on) {
  if (!m) return ALLEGRO_ERR_BAD_ARG;
  cudaStreamSynchronize(m->stream);
  for (auto& r : m->prof_recs) { m->prof_pool.push_back(r.a); m->prof_pool.push_back(r.b); }
  m->prof_recs.clear();
  m->prof = (on & 1) != 0;
  m->nvtx = (on & 2) != 0;
  m->config_gen++;
  return ALLEGRO_OK;
}

extern "C" int allegro_profile_read(allegro_model* m, const char* name, double* ms, int64_t* launches) {
  if (!m || !name || !ms || !launches) return ALLEGRO_ERR_BAD_ARG;
  int cat = -1;
  for (int k = 0; k < PC_COUNT; ++k) if (std::string(name) == kProfNames[k]) cat = k;
  if (cat < 0) { al_set_error(m, "unknown profile group"); return ALLEGRO_ERR_BAD_ARG; }
  AL_CUDA(m, cudaStreamSynchronize(m->stream));
  double tot = 0; int64_t cnt = 0;
  for (auto& r : m->prof_recs)
    if (r.cat == cat) { float t = 0; cudaEventElapsedTime(&t, r.a, r.b); tot += t; cnt++; }
  *ms = tot; *launches = cnt;
  return ALLEGRO_OK;
}
