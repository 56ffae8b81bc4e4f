/* oracle/ovr.h — C interface of the CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, single-threaded ray caster written from BASELINE.json `north_star` and the
 * readings O-1 ... O-12 of SURVEY.md section 8(c) (PAPER.md itself only says "using the
 * ray-casting algorithm", line 13 Abstract; "colour map", line 31 section 2; "orientation
 * information ... output size (defined by the user)", lines 37-45 section 3; float32 voxels,
 * line 57 footnote 4).  It shares no code with the CUDA path under paper_1012_2909_b200/csrc and
 * may be imported only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs.
 */
#ifndef OVR_H
#define OVR_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* Cube storage handed to the oracle: a table of PLAIN bricks (no halo), brick b =
 * bx_i + gx*(by_i + gy*bz_i), each holding its clipped extent ex*ey*ez x-fastest.  A NULL
 * entry means "not resident"; touching it is an error (OVR_ERR_MISSING).  A linear cube is the
 * one-brick case bx=nx, by=ny, bz=nz.  This is storage only: no computation is blocked by it. */
typedef struct {
    int nx, ny, nz;
    int bx, by, bz;
    const float* const* bricks;
} ovr_volume;

typedef struct {
    float m[16];      /* row-major, clip = M (x,y,z,1)^T, voxel coordinates, GL clip space (O-2) */
    int width, height;
    float step;       /* Delta, voxels (O-3) */
} ovr_view;

typedef struct {
    float rgba[256 * 4]; /* (r,g,b,a); a = opacity per unit voxel length (O-6) */
    float vmin, vmax;
} ovr_tf;

enum { OVR_MIP = 0, OVR_EA = 1 };
enum { OVR_F64 = 64, OVR_F32 = 32 };
/* O-8: how a brick partition enters the result */
enum { OVR_UNSPLIT = 0, OVR_SPLIT_GLOBAL = 1, OVR_SPLIT_SORTLAST = 2 };
enum { OVR_OK = 0, OVR_ERR_ARG = -1, OVR_ERR_MISSING = -2, OVR_ERR_SINGULAR = -3 };

typedef struct {
    int mode;          /* OVR_MIP / OVR_EA */
    int precision;     /* OVR_F64 (truth) / OVR_F32 (canonical float32 arithmetic, O-11) */
    int split;         /* OVR_UNSPLIT / OVR_SPLIT_GLOBAL / OVR_SPLIT_SORTLAST */
    int pbx, pby, pbz; /* partition brick size for split != UNSPLIT */
    float tau;         /* ERT threshold; > 1 disables (O-7) */
    float bg[4];       /* background (EA) */
    float miss;        /* MIP value for rays with no taken sample (O-5) */
    int brute;         /* 1: test every lattice k in [0, kmax] (the definition); 0: bracket first */
} ovr_params;

typedef struct {
    int64_t nominal;     /* lattice samples inside the volume (O-3) */
    int64_t taken;       /* samples actually composited (after ERT) */
    int64_t terminated;  /* rays stopped by ERT */
    int64_t flagged;     /* knife-edge pixels (O-12) */
} ovr_counters;

/* Render `n` pixels.  pixels = n x 2 ints (i = column, j = row, row 0 on top) or NULL for the
 * full frame in row-major order (then n must be width*height).  out: EA -> n x 4 floats; MIP ->
 * n floats.  flags (may be NULL): n bytes, 1 = knife-edge pixel (O-12). */
int ovr_render(const ovr_volume* vol, const ovr_view* view, const ovr_tf* tf,
               const ovr_params* prm, const int* pixels, int64_t n,
               float* out, uint8_t* flags, ovr_counters* counters);

/* Sort-last partial image of ONE partition brick (O-8 SORT-LAST): premultiplied (C_b, A_b) with
 * local ERT (EA, 4 floats/pixel) or max / -inf (MIP, 1 float/pixel) over the screen rectangle
 * (x0, y0, w, h), row-major in `out`. */
int ovr_render_brick(const ovr_volume* vol, const ovr_view* view, const ovr_tf* tf,
                     const ovr_params* prm, int brick_id, int x0, int y0, int w, int h,
                     float* out);

/* Fold partial images in the given order (O-8): EA over-operator front to back then background;
 * MIP max then miss value.  rects = n x 4 ints (x0,y0,w,h); partials[i] row-major w*h pixels. */
int ovr_composite(int mode, int precision, int n, const int* rects, const float* const* partials,
                  const int* order, int width, int height, const float* bg, float miss,
                  float* out);

/* O-9 visibility keys of every brick of the grid (gx,gy,gz) of bricks (bx,by,bz); smaller key =
 * closer to the eye.  *is_perspective receives the projection type. */
int ovr_visibility_keys(const ovr_view* view, int bx, int by, int bz, int gx, int gy, int gz,
                        int* keys, int* is_perspective);

/* O-2 ray of pixel (i, j): origin on the near plane, unit direction, length to the far plane. */
int ovr_ray(const ovr_view* view, int i, int j, double o[3], double d[3], double* L);

/* Screen rectangle (x0,y0,w,h) covering every pixel whose ray can hit brick `brick_id`, and the
 * list of partition bricks touched by the rays of the given pixels (marks touched[b] = 1). */
int ovr_bricks_touched(const ovr_view* view, int nx, int ny, int nz, int bx, int by, int bz,
                       const int* pixels, int64_t n, uint8_t* touched);

/* O-6: opacity-corrected table a'_i = 1 - (1 - a_i)^Delta (fp64, rounded to f32). */
int ovr_bake_tf(const ovr_tf* tf, float step, float* baked_rgba);
/* O-6 lookup of one value through the baked (baked=1) or raw table, fp64. */
int ovr_tf_lookup(const ovr_tf* tf, float step, int baked, double v, double rgba[4]);

/* Synthetic cube generator, evaluated in fp64 and rounded to f32, over the
 * voxel box [x0,x0+wx) x [y0,y0+wy) x [z0,z0+wz) of an (nx,ny,nz) cube; out is x-fastest.
 * sources: n_src x 16 doubles (workloads.SRC_COLS); zero_boxes: n_zero x 6 ints inclusive. */
int ovr_generate(uint64_t seed, int nx, int ny, int nz, int x0, int y0, int z0, int wx, int wy,
                 int wz, const double* sources, int n_src, const int* zero_boxes, int n_zero,
                 double continuum, float* out);
/* The N(0,1) noise value of linear voxel index idx (fp64). */
double ovr_noise(uint64_t seed, uint64_t idx);


/* O-14 catalogue overlay (section 2: a source finder's catalogue is "a set
 * of detected astronomical sources represented by their bounding cubes ... superimposed as
 * wireframe boxes on the volume rendering output", moving with the view, selectable, with groups
 * shown / hidden).  boxes = n x 6 ints (xlo xhi ylo yhi zlo zhi, voxel coordinates, inclusive);
 * visible = n bytes or NULL (all shown).  pick = width*height ints, row-major, row 0 on top:
 * 0 where no edge passes, else 1 + the HIGHEST id of the boxes whose wireframe covers the pixel.
 * Rule (O-14): the 12 edges of every shown box are projected with M in fp64, clipped in
 * clip space to w >= 1e-9, |z| <= w and a guard band |x|,|y| <= 2w, mapped to pixel coordinates
 * px = (xn+1) W/2 - 1/2, py = (1-yn) H/2 - 1/2 and sampled at n+1 equidistant points,
 * n = max(1, ceil(max(|dpx|,|dpy|))), each rounded to the nearest pixel (floor(v + 1/2)). */
int ovr_overlay(const ovr_view* view, const int* boxes, int n, const uint8_t* visible, int32_t* pick);
/* The box to select for a click at pixel (x, y): among the covered pixels of the square window of
 * half-width `radius` the one at the smallest Euclidean distance (ties: the larger id); -1 if none. */
int ovr_overlay_pick(const int32_t* pick, int width, int height, int x, int y, int radius);

#ifdef __cplusplus
}
#endif
#endif
