/*
 * dloc_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, obviously-correct CPU implementation (fp64) of the network the PAPER itself
 * describes, as opposed to the residual stack BASELINE.json fixes
 * (smlm_oracle.c).  Only tests/ may build, load or call this file; it shares no code,
 * header, table or helper with the CUDA library under paper_2410_02314_b200/ (nor with
 * smlm_oracle.c) and neither includes the other.
 *
 * What the paper fixes (PAPER.md = /root/reference/PAPER.md, "P:nn" = line nn):
 *   P:57  "the Dense Connection Dilated Block (DCD), which combines dense connections with
 *          dilated convolutions"; "Dense connections allow each layer to utilize outputs
 *          from all preceding layers";
 *   P:59  "Coarse-Grained Sampling, consists of n=1 DCD, and ... Multi-Scale Context
 *          Aggregation, is composed of n=3 DCDs";
 *   P:144 "The current dilation parameters used in this paper are (2, 4, 8, 16)";
 *   P:61  "fine-grained processing using a two-stage U-Net"; P:192(2) "uses two upsampling
 *          stages"; "each pixel outputs the probability of a fluorescent molecule, along with
 *          the offset and uncertainty of the fluorescent molecule's position relative to that
 *          pixel" (DECODE-style heads);
 *   P:53  DECODE "improves localization accuracy using contextual three-frame information"
 *          (the optional 3-frame input).
 * The paper gives no widths, no growth rate, no kernel sizes, no pooling rule and no head
 * activations (Figure 2 is a picture).  Every such number is a READING, listed as D1-D9 in
 * DESIGN.md and restated at the function that uses it.  The net is an exact deterministic
 * function, so this file is the definition written out: no blocking, fusion or reordering.
 *
 * Pins (tests/test_dloc_oracle_pins.py): torch.nn.functional conv2d / max_pool2d /
 * interpolate in fp64 layer by layer, brute-force scatter-form convolution over concatenated
 * inputs, zero-input -> bias-only, hand-computed tiny cases of pooling / up-sampling /
 * uncertainty decode.  The paper prints no worked example, so numerical parity WITH THE
 * PAPER is unpinned.
 *
 * Layout: feature maps planar [c][y][x] as double; weights come in as the caller's fp32 blob
 * (OIHW, cross-correlation) and are widened to double.  Summation order inside one output
 * value is fixed (ci, ky, kx ascending); OpenMP over output channels only.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define DLOC_HEADS 10 /* p, dx, dy, z, N, bg, sigma_x, sigma_y, sigma_z, sigma_N (reading D7) */

typedef struct {
  int32_t c0;        /* base width C0 (reading D1) */
  int32_t growth;    /* G: channels each DCD layer adds (reading D1) */
  int32_t n_blocks;  /* 1 coarse + 3 context = 4 */
  int32_t n_dil;     /* layers per DCD = number of dilations */
  int32_t dilations[8]; /* (2, 4, 8, 16) */
  int32_t in_frames; /* 1, or 3: frames f-1, f, f+1 as stem input channels (reading D8) */
  int32_t stem_relu;
  double norm_scale;
} dloc_net;

typedef struct {
  double pixel_size_nm;
  double offset, gain;
  const float *offset_map; /* [H][W] or NULL */
  const float *gain_map;
} dloc_camera;

/* blob: stem W[C0][in][3][3] b[C0]; per block: per layer i W[G][C0+iG][3][3] b[G], then the
 * transition W[C0][C0+nG][1][1] b[C0]; U-Net enc1 W[2C0][C0][3][3] b, enc2 W[4C0][2C0][3][3] b,
 * dec1 W[2C0][6C0][3][3] b, dec0 W[C0][3C0][3][3] b; heads W[10][C0] b[10]. */
int64_t dloc_oracle_blob_size(const dloc_net *n) {
  int64_t C = n->c0, G = n->growth, s = 0;
  s += C * n->in_frames * 9 + C;
  for (int b = 0; b < n->n_blocks; ++b) {
    for (int i = 0; i < n->n_dil; ++i) s += G * (C + i * G) * 9 + G;
    s += C * (C + n->n_dil * G) + C;
  }
  s += 2 * C * C * 9 + 2 * C;
  s += 4 * C * 2 * C * 9 + 4 * C;
  s += 2 * C * 6 * C * 9 + 2 * C;
  s += C * 3 * C * 9 + C;
  s += DLOC_HEADS * C + DLOC_HEADS;
  return s;
}

/* out[co][y][x] = act(b[co] + sum_{ci,ky,kx} w[co][ci][ky][kx] * in[ci][y+(ky-r)d][x+(kx-r)d]),
 * k = 2r+1 in {1, 3}, out-of-frame := 0 ("same" zero padding, reading D2), act = ReLU iff relu. */
static void conv(const double *in, int cin, int H, int W, const float *w, const float *b, int cout, int k,
                 int d, int relu, double *out) {
  const int r = k / 2;
#pragma omp parallel for schedule(static)
  for (int co = 0; co < cout; ++co)
    for (int y = 0; y < H; ++y)
      for (int x = 0; x < W; ++x) {
        double acc = (double)b[co];
        for (int ci = 0; ci < cin; ++ci)
          for (int ky = 0; ky < k; ++ky)
            for (int kx = 0; kx < k; ++kx) {
              int yy = y + (ky - r) * d, xx = x + (kx - r) * d;
              if (yy < 0 || yy >= H || xx < 0 || xx >= W) continue;
              acc += (double)w[(((int64_t)co * cin + ci) * k + ky) * k + kx] * in[((int64_t)ci * H + yy) * W + xx];
            }
        if (relu && acc < 0.0) acc = 0.0;
        out[((int64_t)co * H + y) * W + x] = acc;
      }
}

/* 2x2 max pooling, stride 2, floor: Ho = H/2, Wo = W/2 (a trailing odd row/column is dropped; D4). */
static void maxpool2(const double *in, int c, int H, int W, double *out) {
  int Ho = H / 2, Wo = W / 2;
  for (int ch = 0; ch < c; ++ch)
    for (int y = 0; y < Ho; ++y)
      for (int x = 0; x < Wo; ++x) {
        const double *p = in + ((int64_t)ch * H + 2 * y) * W + 2 * x;
        double m = p[0];
        if (p[1] > m) m = p[1];
        if (p[W] > m) m = p[W];
        if (p[W + 1] > m) m = p[W + 1];
        out[((int64_t)ch * Ho + y) * Wo + x] = m;
      }
}

/* nearest-neighbour up-sampling by 2 to exactly Ho x Wo: out[y][x] = in[min(y/2, H-1)][min(x/2, W-1)] (D5). */
static void upsample2(const double *in, int c, int H, int W, int Ho, int Wo, double *out) {
  for (int ch = 0; ch < c; ++ch)
    for (int y = 0; y < Ho; ++y)
      for (int x = 0; x < Wo; ++x) {
        int ys = y / 2 < H - 1 ? y / 2 : H - 1, xs = x / 2 < W - 1 ? x / 2 : W - 1;
        out[((int64_t)ch * Ho + y) * Wo + x] = in[((int64_t)ch * H + ys) * W + xs];
      }
}

/* Test hooks: the two resampling rules on their own, so that tests/test_dloc_oracle_pins.py can
 * pin them to a library routine and to hand-written cases (they add no arithmetic). */
int dloc_oracle_maxpool2(const double *in, int c, int H, int W, double *out) {
  if (!in || !out || c < 1 || H < 2 || W < 2) return -1;
  maxpool2(in, c, H, W, out);
  return 0;
}
int dloc_oracle_upsample2(const double *in, int c, int H, int W, int Ho, int Wo, double *out) {
  if (!in || !out || c < 1 || H < 1 || W < 1 || Ho < 1 || Wo < 1) return -1;
  upsample2(in, c, H, W, Ho, Wo, out);
  return 0;
}

/*
 * Forward pass for n frames of H x W uint16 (H, W >= 4).  out_maps [n][10][H][W]: the
 * PRE-activation head outputs.  dump (may be NULL) receives, per frame, the feature maps in
 * this order, each planar [c][h][w]:  stem (C0,H,W); after each block its transition output
 * (C0,H,W) x n_blocks; e1 (2C0,H/2,W/2); e2 (4C0,H/4,W/4); m1 (2C0,H/2,W/2); m0 (C0,H,W).
 * Returns 0 or -1.
 */
int dloc_oracle_forward_maps(const dloc_net *net, const float *weights, const uint16_t *frames, int64_t n,
                             int H, int W, const dloc_camera *cam, double *out_maps, double *dump) {
  if (!net || !weights || !frames || !cam || !out_maps) return -1;
  const int C = net->c0, G = net->growth, NB = net->n_blocks, ND = net->n_dil, IF = net->in_frames;
  if (C < 1 || G < 1 || NB < 1 || ND < 1 || ND > 8 || (IF != 1 && IF != 3) || H < 4 || W < 4) return -1;
  const int64_t px = (int64_t)H * W;
  const int H2 = H / 2, W2 = W / 2, H4 = H2 / 2, W4 = W2 / 2;
  const int CB = C + ND * G;
  double *xin = (double *)malloc(sizeof(double) * IF * px);
  double *blk = (double *)malloc(sizeof(double) * CB * px);      /* f_0 | g_0 | g_1 ... (the dense concatenation) */
  double *e0 = (double *)malloc(sizeof(double) * C * px);
  double *p1 = (double *)malloc(sizeof(double) * C * H2 * W2);
  double *cat1 = (double *)malloc(sizeof(double) * 6 * C * H2 * W2);  /* up(e2) | e1 */
  double *p2 = (double *)malloc(sizeof(double) * 2 * C * H4 * W4);
  double *e2 = (double *)malloc(sizeof(double) * 4 * C * H4 * W4);
  double *m1 = (double *)malloc(sizeof(double) * 2 * C * H2 * W2);
  double *cat0 = (double *)malloc(sizeof(double) * 3 * C * px);       /* up(m1) | e0 */
  double *m0 = (double *)malloc(sizeof(double) * C * px);
  if (!xin || !blk || !e0 || !p1 || !cat1 || !p2 || !e2 || !m1 || !cat0 || !m0) return -1;
  for (int64_t f = 0; f < n; ++f) {
    const float *wp = weights;
    double *dp = dump ? dump + f * ((int64_t)(1 + NB) * C * px + (int64_t)4 * C * H2 * W2 + (int64_t)4 * C * H4 * W4 +
                                    (int64_t)C * px)
                      : NULL;
    /* input: xhat = ((adu - offset) / gain) / norm_scale per frame; with in_frames = 3 the
     * channels are frames f-1, f, f+1, indices clamped to [0, n-1] (reading D8) */
    for (int ch = 0; ch < IF; ++ch) {
      int64_t g = IF == 1 ? f : f + ch - 1;
      if (g < 0) g = 0;
      if (g > n - 1) g = n - 1;
      for (int64_t i = 0; i < px; ++i) {
        double off = cam->offset_map ? (double)cam->offset_map[i] : cam->offset;
        double gain = cam->gain_map ? (double)cam->gain_map[i] : cam->gain;
        xin[ch * px + i] = (((double)frames[g * px + i] - off) / gain) / net->norm_scale;
      }
    }
    /* stem: 3x3, in_frames -> C0 */
    conv(xin, IF, H, W, wp, wp + (int64_t)C * IF * 9, C, 3, 1, net->stem_relu, blk);
    wp += (int64_t)C * IF * 9 + C;
    if (dp) { memcpy(dp, blk, sizeof(double) * C * px); dp += C * px; }
    /* DCD blocks: layer i sees the concatenation of the block input and of the
     * outputs of layers 0..i-1 and adds G channels (3x3, dilation d_i, ReLU); a 1x1
     * transition (ReLU) brings the C0 + n G channels back to C0 (readings D1, D3) */
    for (int b = 0; b < NB; ++b) {
      for (int i = 0; i < ND; ++i) {
        int cin = C + i * G;
        conv(blk, cin, H, W, wp, wp + (int64_t)G * cin * 9, G, 3, net->dilations[i], 1, blk + (int64_t)cin * px);
        wp += (int64_t)G * cin * 9 + G;
      }
      conv(blk, CB, H, W, wp, wp + (int64_t)C * CB, C, 1, 1, 1, e0);
      wp += (int64_t)C * CB + C;
      if (dp) { memcpy(dp, e0, sizeof(double) * C * px); dp += C * px; }
      memcpy(blk, e0, sizeof(double) * C * px);
    }
    /* two-stage U-Net (P:61, P:192(2); readings D4-D6): widths C0, 2C0, 4C0 */
    maxpool2(e0, C, H, W, p1);
    double *e1 = cat1 + (int64_t)4 * C * H2 * W2;
    conv(p1, C, H2, W2, wp, wp + (int64_t)2 * C * C * 9, 2 * C, 3, 1, 1, e1);
    wp += (int64_t)2 * C * C * 9 + 2 * C;
    if (dp) { memcpy(dp, e1, sizeof(double) * 2 * C * H2 * W2); dp += (int64_t)2 * C * H2 * W2; }
    maxpool2(e1, 2 * C, H2, W2, p2);
    conv(p2, 2 * C, H4, W4, wp, wp + (int64_t)4 * C * 2 * C * 9, 4 * C, 3, 1, 1, e2);
    wp += (int64_t)4 * C * 2 * C * 9 + 4 * C;
    if (dp) { memcpy(dp, e2, sizeof(double) * 4 * C * H4 * W4); dp += (int64_t)4 * C * H4 * W4; }
    upsample2(e2, 4 * C, H4, W4, H2, W2, cat1);
    conv(cat1, 6 * C, H2, W2, wp, wp + (int64_t)2 * C * 6 * C * 9, 2 * C, 3, 1, 1, m1);
    wp += (int64_t)2 * C * 6 * C * 9 + 2 * C;
    if (dp) { memcpy(dp, m1, sizeof(double) * 2 * C * H2 * W2); dp += (int64_t)2 * C * H2 * W2; }
    upsample2(m1, 2 * C, H2, W2, H, W, cat0);
    memcpy(cat0 + (int64_t)2 * C * px, e0, sizeof(double) * C * px);
    conv(cat0, 3 * C, H, W, wp, wp + (int64_t)C * 3 * C * 9, C, 3, 1, 1, m0);
    wp += (int64_t)C * 3 * C * 9 + C;
    if (dp) { memcpy(dp, m0, sizeof(double) * C * px); dp += C * px; }
    /* heads: 1x1, C0 -> 10, no activation here */
    conv(m0, C, H, W, wp, wp + (int64_t)DLOC_HEADS * C, DLOC_HEADS, 1, 1, 0, out_maps + f * DLOC_HEADS * px);
  }
  free(xin); free(blk); free(e0); free(p1); free(cat1); free(p2); free(e2); free(m1); free(cat0); free(m0);
  return 0;
}

/* Uncertainty heads at given pixels (reading D7, DECODE-style bounded positive outputs):
 *   sigma_x_nm = sigma_xy_px * sigmoid(o_6) * pixel_size,  sigma_y likewise (o_7),
 *   sigma_z_nm = sigma_z_nm_scale * sigmoid(o_8),  sigma_N = sigma_n_scale * sigmoid(o_9).
 * o [n][10][H][W]; (frame, pix)[count] -> out[count][4]. */
static double sigmoid_(double v) {
  if (v >= 0.0) return 1.0 / (1.0 + exp(-v));
  double e = exp(v);
  return e / (1.0 + e);
}
int dloc_oracle_sigmas(const double *o, int H, int W, const int32_t *frame, const int32_t *pix, int64_t count,
                       double pixel_size_nm, double sigma_xy_px, double sigma_z_scale_nm, double sigma_n_scale,
                       double *out) {
  if (!o || !frame || !pix || !out) return -1;
  int64_t px = (int64_t)H * W;
  for (int64_t i = 0; i < count; ++i) {
    const double *m = o + (int64_t)frame[i] * DLOC_HEADS * px + pix[i];
    out[4 * i + 0] = sigma_xy_px * sigmoid_(m[6 * px]) * pixel_size_nm;
    out[4 * i + 1] = sigma_xy_px * sigmoid_(m[7 * px]) * pixel_size_nm;
    out[4 * i + 2] = sigma_z_scale_nm * sigmoid_(m[8 * px]);
    out[4 * i + 3] = sigma_n_scale * sigmoid_(m[9 * px]);
  }
  return 0;
}
