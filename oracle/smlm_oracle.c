/*
 * smlm_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64) of the one hot path of
 * arXiv 2410.02314 that BASELINE.json `north_star` names:
 *
 *   uint16 frames -> normalise -> 3x3 stem conv -> L dilated 3x3 conv layers
 *   (ReLU + residual) -> 1x1 heads -> sigmoid / threshold / 3x3 local-maximum
 *   suppression / sub-pixel decode -> emitter list.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference`
 * leg may build, load or call this file.  It shares no code, header, table or helper
 * with the CUDA library under paper_2410_02314_b200/ and neither includes the other.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md, "P:nn" = line nn):
 *   - the network is a stack of dilated convolutions (dilation set P:144) whose
 *     per-pixel outputs are "the probability of a fluorescent molecule, along with the
 *     offset ... of the fluorescent molecule's position relative to that pixel";
 *   - post-processing converts "these offsets into absolute coordinates" (P:192 item 3)
 *     and runs on the GPU.
 * The paper gives no equation, width or detection rule for inference; all of those come
 * from BASELINE.json `north_star` / `configs` and from the readings G1-G17 listed in
 * DESIGN.md (taken from SURVEY.md section 8(c)).  Each function below cites its step
 * O1..O8 of that list.  The method is an exact deterministic function, so this file is
 * "the definition written out": no blocking, fusion or reordering.
 *
 * Pins (tests/test_oracle_pins.py): brute-force scatter-form convolution on tiny inputs,
 * torch.nn.functional.conv2d in fp64, hand-derived emitter lists for hand-placed delta
 * maps (tests/golden/), and invariants (zero input -> bias only, shift equivariance,
 * identity / single-tap trunks, threshold monotonicity).  The paper prints no worked
 * example for this path, so numerical parity WITH THE PAPER is unpinned.
 *
 * Layout: activations [y][x][c] (channel fastest) as double; weights come in as the
 * caller's fp32 blob (OIHW, cross-correlation, reading G2) and are widened to double.
 * Threads: OpenMP over output rows only; the summation order inside one output value is
 * fixed (ky, kx, ci ascending), so results do not depend on the thread count.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_MAX_LAYERS 32

typedef struct {
  int32_t channels;      /* C */
  int32_t n_layers;      /* L */
  int32_t dilations[ORACLE_MAX_LAYERS];
  int32_t head_channels; /* 5: p,dx,dy,N,bg   6: p,dx,dy,z,N,bg  (reading G6) */
  int32_t stem_relu;     /* reading G3 */
  double norm_scale;     /* 1000 */
  double xy_scale;       /* 0.5 */
  double z_scale_nm;     /* 700 */
  double photon_scale;   /* reading G6 */
  double bg_scale;       /* reading G6 */
  int32_t in_frames;     /* 0 or 1: one frame per input; 3: temporal context, the stem sees the frames
                            f-1, f, f+1 as three input channels ("contextual three-frame
                            information"; reading G24 in DESIGN.md: indices
                            clamped to [0, n-1] of the call) */
} oracle_net;

typedef struct {
  double pixel_size_nm;
  double offset, gain;     /* scalars, used where the maps are NULL */
  const float *offset_map; /* [H][W] or NULL */
  const float *gain_map;   /* [H][W] or NULL */
} oracle_camera;

typedef struct {
  int32_t frame;
  int32_t pix; /* iy * W + ix */
  double x_nm, y_nm, z_nm, photons, bg, p;
} oracle_emitter;

int smlm_oracle_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

static int in_frames_of(const oracle_net *net) { return net->in_frames == 3 ? 3 : 1; }

int64_t smlm_oracle_blob_size(const oracle_net *net) {
  int64_t C = net->channels, L = net->n_layers, nh = net->head_channels, IF = in_frames_of(net);
  return (C * IF * 9 + C) + L * (C * C * 9 + C) + (nh * C + nh);
}

/* O1 normalise: xhat = ((adu - offset) / gain) / norm_scale  (reading G5). */
static void normalise(const uint16_t *frame, int H, int W, const oracle_camera *cam,
                      double norm_scale, double *xhat) {
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      int64_t i = (int64_t)y * W + x;
      double off = cam->offset_map ? (double)cam->offset_map[i] : cam->offset;
      double gain = cam->gain_map ? (double)cam->gain_map[i] : cam->gain;
      xhat[i] = (((double)frame[i] - off) / gain) / norm_scale;
    }
}

/* O2 stem: a0[y,x,co] = act(b0[co] + sum_{ch,ky,kx} W0[co,ch,ky,kx] * xhat[ch][y+ky-1, x+kx-1]),
 * out-of-frame xhat := 0; act = ReLU iff stem_relu (reading G3); ch < IF input channels
 * (IF = 1: the frame itself; IF = 3: the normalised frames f-1, f, f+1, reading G24). */
static void stem(const double *xhat /*[IF][H][W]*/, int IF, int H, int W, int C,
                 const float *w /*[C][IF][3][3]*/, const float *b, int relu, double *a0 /*[H][W][C]*/) {
#pragma omp parallel for schedule(static)
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x)
      for (int co = 0; co < C; ++co) {
        double acc = (double)b[co];
        for (int ch = 0; ch < IF; ++ch)
          for (int ky = 0; ky < 3; ++ky)
            for (int kx = 0; kx < 3; ++kx) {
              int yy = y + ky - 1, xx = x + kx - 1;
              if (yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
              acc += (double)w[((co * IF + ch) * 3 + ky) * 3 + kx] * xhat[((int64_t)ch * H + yy) * W + xx];
            }
        if (relu && acc < 0.0) acc = 0.0;
        a0[((int64_t)y * W + x) * C + co] = acc;
      }
}

/* O3 one trunk layer:
 *   t[y,x,co] = b[co] + sum_{ky,kx,ci} W[co,ci,ky,kx] * a[y+(ky-1)d, x+(kx-1)d, ci]
 *   (out-of-frame := 0, i.e. zero padding = dilation, in the activation domain, G2)
 *   out = a + max(t, 0)                                   (reading G4)
 * `wt` is the layer's weights re-indexed [ky][kx][ci][co] as double so that the
 * innermost loop runs over co; the order of additions into one output value is
 * (ky, kx, ci) ascending. */
static void trunk_layer(const double *a, int H, int W, int C, int d, const double *wt,
                        const float *b, double *out) {
#pragma omp parallel for schedule(static)
  for (int y = 0; y < H; ++y) {
    double acc[256];
    for (int x = 0; x < W; ++x) {
      for (int co = 0; co < C; ++co) acc[co] = (double)b[co];
      for (int ky = 0; ky < 3; ++ky) {
        int yy = y + (ky - 1) * d;
        if (yy < 0 || yy >= H) continue;
        for (int kx = 0; kx < 3; ++kx) {
          int xx = x + (kx - 1) * d;
          if (xx < 0 || xx >= W) continue;
          const double *ain = a + ((int64_t)yy * W + xx) * C;
          const double *wk = wt + (int64_t)(ky * 3 + kx) * C * C;
          for (int ci = 0; ci < C; ++ci) {
            double v = ain[ci];
            const double *wr = wk + (int64_t)ci * C;
            for (int co = 0; co < C; ++co) acc[co] += v * wr[co];
          }
        }
      }
      const double *res = a + ((int64_t)y * W + x) * C;
      double *o = out + ((int64_t)y * W + x) * C;
      for (int co = 0; co < C; ++co) o[co] = res[co] + (acc[co] > 0.0 ? acc[co] : 0.0);
    }
  }
}

/* O4 heads: o[h,y,x] = bh[h] + sum_c Wh[h,c] * aL[y,x,c]. */
static void heads(const double *aL, int H, int W, int C, int nh, const float *wh, const float *bh,
                  double *o /*[nh][H][W]*/) {
#pragma omp parallel for schedule(static)
  for (int y = 0; y < H; ++y)
    for (int x = 0; x < W; ++x) {
      const double *a = aL + ((int64_t)y * W + x) * C;
      for (int h = 0; h < nh; ++h) {
        double acc = (double)bh[h];
        for (int c = 0; c < C; ++c) acc += (double)wh[h * C + c] * a[c];
        o[((int64_t)h * H + y) * W + x] = acc;
      }
    }
}

/*
 * O1-O4 for n frames.  out_maps: [n][n_h][H][W] PRE-activation head outputs o.
 * trunk_dump (may be NULL): [n][L+1][H][W][C], a_0 .. a_L of every frame (debug aid for
 * layer-by-layer comparison).  Returns 0, or -1 on bad arguments / allocation failure.
 */
int smlm_oracle_forward_maps(const oracle_net *net, const float *weights, const uint16_t *frames,
                             int64_t n, int H, int W, const oracle_camera *cam, double *out_maps,
                             double *trunk_dump) {
  if (!net || !weights || !frames || !cam || !out_maps) return -1;
  int C = net->channels, L = net->n_layers, nh = net->head_channels;
  if (C < 1 || C > 256 || L < 0 || L > ORACLE_MAX_LAYERS || (nh != 5 && nh != 6) || H < 1 || W < 1)
    return -1;
  int64_t px = (int64_t)H * W;
  const int IF = in_frames_of(net);
  double *xhat = (double *)malloc(sizeof(double) * px * IF);
  double *a = (double *)malloc(sizeof(double) * px * C);
  double *a2 = (double *)malloc(sizeof(double) * px * C);
  double *wt = (double *)malloc(sizeof(double) * 9 * C * C);
  if (!xhat || !a || !a2 || !wt) {
    free(xhat); free(a); free(a2); free(wt);
    return -1;
  }
  for (int64_t f = 0; f < n; ++f) {
    const float *wp = weights;
    for (int ch = 0; ch < IF; ++ch) { /* IF = 3: frames f-1, f, f+1, clamped to the call (G24) */
      int64_t g = IF == 1 ? f : f + ch - 1;
      if (g < 0) g = 0;
      if (g > n - 1) g = n - 1;
      normalise(frames + g * px, H, W, cam, net->norm_scale, xhat + ch * px);
    }
    stem(xhat, IF, H, W, C, wp, wp + C * IF * 9, net->stem_relu, a);
    wp += C * IF * 9 + C;
    if (trunk_dump) memcpy(trunk_dump + (f * (L + 1) + 0) * px * C, a, sizeof(double) * px * C);
    for (int l = 0; l < L; ++l) {
      /* OIHW [co][ci][ky][kx] -> [ky][kx][ci][co] */
      for (int co = 0; co < C; ++co)
        for (int ci = 0; ci < C; ++ci)
          for (int ky = 0; ky < 3; ++ky)
            for (int kx = 0; kx < 3; ++kx)
              wt[((int64_t)(ky * 3 + kx) * C + ci) * C + co] =
                  (double)wp[(((int64_t)co * C + ci) * 3 + ky) * 3 + kx];
      trunk_layer(a, H, W, C, net->dilations[l], wt, wp + (int64_t)C * C * 9, a2);
      double *t = a; a = a2; a2 = t;
      wp += (int64_t)C * C * 9 + C;
      if (trunk_dump) memcpy(trunk_dump + (f * (L + 1) + l + 1) * px * C, a, sizeof(double) * px * C);
    }
    heads(a, H, W, C, nh, wp, wp + nh * C, out_maps + f * nh * px);
  }
  free(xhat); free(a); free(a2); free(wt);
  return 0;
}

/* O5 activations.  softplus(v) = max(v,0) + log1p(exp(-|v|)) (stable form). */
static double sigmoid_(double v) {
  if (v >= 0.0) return 1.0 / (1.0 + exp(-v));
  double e = exp(v);
  return e / (1.0 + e);
}
static double softplus_(double v) { return (v > 0.0 ? v : 0.0) + log1p(exp(-fabs(v))); }

/*
 * O5 on whole maps: in o [n][n_h][H][W] -> out act [n][n_h][H][W], the "raw output maps"
 * of the parity gate: p = sigmoid(o_p); dx,dy = xy_scale*tanh(.) in pixels;
 * z -> tanh(o_z) (dimensionless, before z_scale); N, bg -> softplus(.) (before unit scale).
 */
int smlm_oracle_activate_maps(const oracle_net *net, const double *o, int64_t n, int H, int W,
                              double *act) {
  if (!net || !o || !act) return -1;
  int nh = net->head_channels;
  int64_t px = (int64_t)H * W;
  for (int64_t f = 0; f < n; ++f)
    for (int h = 0; h < nh; ++h) {
      const double *src = o + (f * nh + h) * px;
      double *dst = act + (f * nh + h) * px;
      int is_z = (nh == 6 && h == 3);
      for (int64_t i = 0; i < px; ++i) {
        if (h == 0) dst[i] = sigmoid_(src[i]);
        else if (h == 1 || h == 2) dst[i] = net->xy_scale * tanh(src[i]);
        else if (is_z) dst[i] = tanh(src[i]);
        else dst[i] = softplus_(src[i]);
      }
    }
  return 0;
}

/*
 * O6-O8 detect + decode + emit, on PRE-activation maps o [n][n_h][H][W].
 *  O6  pixel q is an emitter iff o_p[q] > logit(thr) (p > thr strictly, G9/G10) AND for all
 *      8 neighbours m inside the frame: o_p[q] > o_p[m], or o_p[q] == o_p[m] and
 *      idx(q) < idx(m)  (single pass on the raw logits; lower index wins ties; neighbours
 *      outside the frame never win; reading G8).  thr <= 0 -> every local maximum,
 *      thr >= 1 -> none.
 *  O7  x_nm = (ix + dx) * pixel_size, y_nm = (iy + dy) * pixel_size (pixel centres at
 *      integer coordinates, reading G7); z = z_scale*tanh(o_z) if n_h == 6 else 0;
 *      N = photon_scale*softplus(o_N); bg = bg_scale*softplus(o_bg); p = sigmoid(o_p).
 *  O8  records in (frame, pix) ascending order.
 * *count receives the number found; at most `capacity` records are written.
 */
int smlm_oracle_postprocess(const oracle_net *net, const double *o, int64_t n, int H, int W,
                            const oracle_camera *cam, double threshold, oracle_emitter *out,
                            int64_t capacity, int64_t *count) {
  if (!net || !o || !cam || !count) return -1;
  int nh = net->head_channels;
  int64_t px = (int64_t)H * W, found = 0;
  int none = (threshold >= 1.0), all = (threshold <= 0.0);
  double lthr = (none || all) ? 0.0 : log(threshold / (1.0 - threshold));
  for (int64_t f = 0; f < n && !none; ++f) {
    const double *op = o + (f * nh + 0) * px;
    for (int y = 0; y < H; ++y)
      for (int x = 0; x < W; ++x) {
        int64_t q = (int64_t)y * W + x;
        double v = op[q];
        if (!all && !(v > lthr)) continue;
        int is_max = 1;
        for (int dy = -1; dy <= 1 && is_max; ++dy)
          for (int dx = -1; dx <= 1; ++dx) {
            if (dy == 0 && dx == 0) continue;
            int yy = y + dy, xx = x + dx;
            if (yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
            int64_t m = (int64_t)yy * W + xx;
            if (!(v > op[m] || (v == op[m] && q < m))) { is_max = 0; break; }
          }
        if (!is_max) continue;
        if (out && found < capacity) {
          oracle_emitter *e = out + found;
          double odx = o[(f * nh + 1) * px + q], ody = o[(f * nh + 2) * px + q];
          int hN = (nh == 6) ? 4 : 3, hB = hN + 1;
          e->frame = (int32_t)f;
          e->pix = (int32_t)q;
          e->x_nm = ((double)x + net->xy_scale * tanh(odx)) * cam->pixel_size_nm;
          e->y_nm = ((double)y + net->xy_scale * tanh(ody)) * cam->pixel_size_nm;
          e->z_nm = (nh == 6) ? net->z_scale_nm * tanh(o[(f * nh + 3) * px + q]) : 0.0;
          e->photons = net->photon_scale * softplus_(o[(f * nh + hN) * px + q]);
          e->bg = net->bg_scale * softplus_(o[(f * nh + hB) * px + q]);
          e->p = sigmoid_(v);
        }
        ++found;
      }
  }
  *count = found;
  return 0;
}
