/* Plain C99 client of include/trk.h (no Python, no torch, no CUDA headers): the served request of PAPER.md lines 157-160
 * through trk_create / trk_infer_host / trk_infer_host_tracks / trk_destroy with HOST buffers.  Weights and hits are
 * pseudo-random; what is checked are the invariants that hold for any weights: status codes, label = smallest hit index
 * of its component (label[v] <= v, label[label[v]] == label[v]), no label across events, track lists consistent with the
 * labels, identical results on a second call, error statuses for bad arguments.
 * Built and run by tests/test_gpu_c_abi.py:  gcc -std=c99 -I include trk_c_smoke.c -L <pkg> -ltrk -lm  */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "trk.h"

static unsigned long long g_state = 0x9E3779B97F4A7C15ull;
static double uniform(void) { /* xorshift64*, (0,1) */
  g_state ^= g_state >> 12; g_state ^= g_state << 25; g_state ^= g_state >> 27;
  return ((g_state * 0x2545F4914F6CDD1Dull) >> 11) * (1.0 / 9007199254740992.0) + 1e-12;
}

typedef struct { int n; int32_t dims[8]; float* w[8]; float* b[8]; const float* wp[8]; const float* bp[8]; } mlp_store;

static trk_mlp make_mlp(mlp_store* s, int n, const int* dims) {
  s->n = n;
  for (int l = 0; l <= n; ++l) s->dims[l] = dims[l];
  for (int l = 0; l < n; ++l) {
    const int in = dims[l], out = dims[l + 1];
    const double bound = sqrt(6.0 / in);
    s->w[l] = (float*)malloc(sizeof(float) * in * out);
    s->b[l] = (float*)malloc(sizeof(float) * out);
    for (int i = 0; i < in * out; ++i) s->w[l][i] = (float)((2.0 * uniform() - 1.0) * bound);
    for (int i = 0; i < out; ++i) s->b[l][i] = (float)((2.0 * uniform() - 1.0) / sqrt((double)in));
    s->wp[l] = s->w[l];
    s->bp[l] = s->b[l];
  }
  trk_mlp m;
  m.n_layers = n; m.dims = s->dims; m.weight = s->wp; m.bias = s->bp;
  return m;
}

#define CHECK(cond, msg) do { if (!(cond)) { fprintf(stderr, "FAIL: %s (line %d)\n", msg, __LINE__); return 1; } } while (0)

int main(void) {
  enum { H = 64, N0 = 300, N1 = 200, N = N0 + N1 };
  static mlp_store st[7];
  const int d_embed[] = {3, 64, 64, 8}, d_filter[] = {6, 64, 1}, d_nenc[] = {3, H, H}, d_eenc[] = {4, H, H},
            d_enet[] = {3 * H, H, H}, d_nnet[] = {3 * H, H, H}, d_edec[] = {3 * H, H, 1};
  trk_config cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.struct_size = (uint32_t)sizeof(cfg);
  cfg.device = 0;
  cfg.precision = TRK_FP32;
  cfg.embed = make_mlp(&st[0], 3, d_embed);
  cfg.frnn_radius = 0.6f;
  cfg.frnn_k = 16;
  cfg.grid_proj = NULL;
  cfg.grid_dims = 3;
  cfg.filter = make_mlp(&st[1], 2, d_filter);
  cfg.filter_input = TRK_FILTER_RAW;
  cfg.filter_cut = 0.4f;
  cfg.gnn_hidden = H; cfg.gnn_iters = 3; cfg.gnn_layernorm = 1;
  cfg.node_enc = make_mlp(&st[2], 2, d_nenc);
  cfg.edge_enc = make_mlp(&st[3], 2, d_eenc);
  cfg.edge_net = make_mlp(&st[4], 2, d_enet);
  cfg.node_net = make_mlp(&st[5], 2, d_nnet);
  cfg.edge_dec = make_mlp(&st[6], 2, d_edec);
  st[6].b[1][0] += 1.0f; /* centre the random decoder's logits around the cut so that both sides occur */
  cfg.gnn_cut = 0.5f;
  cfg.max_hits = N; cfg.max_events = 2; cfg.max_cand_edges = (int64_t)N * 16; cfg.max_kept_edges = (int64_t)N * 16;
  cfg.min_track_hits = 2;

  /* a wrong struct_size must be refused before anything is allocated */
  trk_ctx* ctx = NULL;
  cfg.struct_size += 4;
  CHECK(trk_create(&cfg, &ctx) == TRK_ERR_INVALID_ARG && ctx == NULL, "struct_size mismatch not refused");
  CHECK(strlen(trk_last_error(NULL)) > 0, "no error text for the failed trk_create");
  cfg.struct_size -= 4;
  trk_status s = trk_create(&cfg, &ctx);
  if (s != TRK_OK) { fprintf(stderr, "trk_create: %s: %s\n", trk_status_string(s), trk_last_error(NULL)); return 1; }
  CHECK(trk_workspace_bytes(ctx) > 0, "workspace size");

  /* two events of hits on ten layers: (r/1000, phi/pi, z/1000) */
  static const float layers[10] = {0.032f, 0.072f, 0.116f, 0.172f, 0.260f, 0.360f, 0.500f, 0.660f, 0.820f, 1.020f};
  static float hits[N][3];
  for (int i = 0; i < N; ++i) {
    hits[i][0] = layers[(int)(uniform() * 10.0) % 10];
    hits[i][1] = (float)(2.0 * uniform() - 1.0);
    hits[i][2] = (float)(2.0 * uniform() - 1.0);
  }
  const int32_t offsets[3] = {0, N0, N};
  static int32_t labels[N], labels2[N], toff[N + 1], thit[N], counts[6], counts4[4];

  s = trk_infer_host(ctx, 2, offsets, &hits[0][0], labels, counts4);
  if (s != TRK_OK) { fprintf(stderr, "trk_infer_host: %s: %s\n", trk_status_string(s), trk_last_error(ctx)); return 1; }
  CHECK(counts4[3] == 0 && counts4[0] > 0 && counts4[1] <= counts4[0] && counts4[2] <= counts4[1], "counts");
  CHECK(trk_last_launch_count(ctx) > 0, "no kernel of the library was launched");
  CHECK(counts4[2] > 0 && counts4[2] < counts4[1], "the GNN cut should have edges on both sides");
  for (int v = 0; v < N; ++v) {
    CHECK(labels[v] >= 0 && labels[v] <= v, "label is not the smallest index of its component");
    CHECK(labels[labels[v]] == labels[v], "label of a label");
    CHECK((v < N0) == (labels[v] < N0), "a component spans two events");
  }

  s = trk_infer_host_tracks(ctx, 2, offsets, &hits[0][0], labels2, toff, thit, counts);
  if (s != TRK_OK) { fprintf(stderr, "trk_infer_host_tracks: %s: %s\n", trk_status_string(s), trk_last_error(ctx)); return 1; }
  CHECK(memcmp(labels, labels2, sizeof(labels)) == 0, "second call gives different labels");
  CHECK(memcmp(counts, counts4, sizeof(counts4)) == 0, "second call gives different counts");
  const int T = counts[4], nh = counts[5];
  CHECK(T >= 0 && toff[0] == 0 && toff[T] == nh && nh <= N, "track offsets");
  int size_of[N];
  memset(size_of, 0, sizeof(size_of));
  for (int v = 0; v < N; ++v) size_of[labels[v]]++;
  int want_tracks = 0, want_hits = 0;
  for (int v = 0; v < N; ++v)
    if (labels[v] == v && size_of[v] >= 2) { want_tracks++; want_hits += size_of[v]; }
  CHECK(T == want_tracks && nh == want_hits, "number of tracks / hits in tracks");
  for (int t = 0; t < T; ++t) {
    const int b = toff[t], e = toff[t + 1];
    CHECK(e - b >= 2 && thit[b] == labels[thit[b]], "a track must start with its label and have min_track_hits hits");
    CHECK(e - b == size_of[thit[b]], "track length != component size");
    for (int k = b; k < e; ++k) {
      CHECK(labels[thit[k]] == thit[b], "hit of another component in a track");
      CHECK(k == b || thit[k] > thit[k - 1], "hits of a track must ascend");
    }
    CHECK(t == 0 || thit[b] > thit[toff[t - 1]], "tracks must ascend by label");
  }

  /* host-detectable errors: nothing is enqueued, the ctx stays usable */
  const int32_t bad_off[3] = {0, N0, N0 - 1};
  CHECK(trk_infer_host(ctx, 2, bad_off, &hits[0][0], labels2, NULL) == TRK_ERR_INVALID_ARG, "non-monotone offsets accepted");
  const int32_t big_off[2] = {0, N + 1};
  CHECK(trk_infer_host(ctx, 1, big_off, &hits[0][0], labels2, NULL) == TRK_ERR_CAPACITY, "N > max_hits accepted");
  CHECK(trk_infer_host(ctx, 2, offsets, NULL, labels2, NULL) == TRK_ERR_INVALID_ARG, "NULL hits accepted");
  s = trk_infer_host(ctx, 2, offsets, &hits[0][0], labels2, counts4);
  CHECK(s == TRK_OK && memcmp(labels, labels2, sizeof(labels)) == 0, "ctx unusable after a refused call");

  CHECK(trk_destroy(ctx) == TRK_OK && trk_destroy(NULL) == TRK_OK, "trk_destroy");
  printf("OK tracks=%d hits_in_tracks=%d E_c=%d E_k=%d E_t=%d\n", T, nh, counts[0], counts[1], counts[2]);
  return 0;
}
