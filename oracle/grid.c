/*
 * grid.c -- CPU ORACLE (test infrastructure): quadtree levels, Morton order, neighbour
 * lists, ghost band and ghost lists (paper Sec. 4.3-4.4, Sec. 3.2 P:94, P:110-114;
 * the concrete rules are the readings listed in DESIGN.md "Grid rules").
 * Technique on purpose different from the product's builder: one open-addressing hash
 * map (ix,iy) -> cell per level, qsort on Morton keys.
 */
#include "internal.h"
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------- hash map */
typedef struct {
  uint64_t* key;
  int32_t* val;
  uint64_t cap, mask;
  int64_t n;
} hmap;

#define HKEY_EMPTY 0xFFFFFFFFFFFFFFFFull
#define CBIAS 1024   /* boundary cells have slightly negative coordinates */

static uint64_t pack_xy(int ix, int iy)
{
  return ((uint64_t)(uint32_t)(ix + CBIAS) << 32) | (uint64_t)(uint32_t)(iy + CBIAS);
}

static uint64_t hash64(uint64_t x)
{
  x ^= x >> 33; x *= 0xff51afd7ed558ccdull; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ull; x ^= x >> 33;
  return x;
}

static int hmap_init(hmap* h, int64_t expected)
{
  uint64_t cap = 16;
  while (cap < (uint64_t)(2 * expected + 8)) cap <<= 1;
  h->cap = cap; h->mask = cap - 1; h->n = 0;
  h->key = (uint64_t*)malloc(cap * sizeof(uint64_t));
  h->val = (int32_t*)malloc(cap * sizeof(int32_t));
  if (!h->key || !h->val) return ORC_ENOMEM;
  memset(h->key, 0xFF, cap * sizeof(uint64_t));
  return ORC_OK;
}
static void hmap_free(hmap* h) { free(h->key); free(h->val); h->key = 0; h->val = 0; }

static int hmap_grow(hmap* h);
static int hmap_put(hmap* h, uint64_t k, int32_t v)
{
  if ((uint64_t)(2 * (h->n + 1)) > h->cap) { int rc = hmap_grow(h); if (rc) return rc; }
  uint64_t p = hash64(k) & h->mask;
  while (h->key[p] != HKEY_EMPTY && h->key[p] != k) p = (p + 1) & h->mask;
  if (h->key[p] == HKEY_EMPTY) { h->key[p] = k; h->n++; }
  h->val[p] = v;
  return ORC_OK;
}
static int hmap_grow(hmap* h)
{
  hmap o = *h;
  int rc = hmap_init(h, (int64_t)o.cap);
  if (rc) return rc;
  for (uint64_t p = 0; p < o.cap; ++p)
    if (o.key[p] != HKEY_EMPTY) hmap_put(h, o.key[p], o.val[p]);
  hmap_free(&o);
  return ORC_OK;
}
/* returns value or -1 */
static int32_t hmap_get(const hmap* h, uint64_t k)
{
  uint64_t p = hash64(k) & h->mask;
  while (h->key[p] != HKEY_EMPTY) {
    if (h->key[p] == k) return h->val[p];
    p = (p + 1) & h->mask;
  }
  return -1;
}

/* ------------------------------------------------------------------ Morton */
/* Z-order key with x in the even bits (bit 0) and y in the odd bits (reading S5) */
static uint64_t morton(uint32_t x, uint32_t y)
{
  uint64_t k = 0;
  for (int b = 0; b < 32; ++b) {
    k |= (uint64_t)((x >> b) & 1u) << (2 * b);
    k |= (uint64_t)((y >> b) & 1u) << (2 * b + 1);
  }
  return k;
}

typedef struct { uint64_t key; int32_t ix, iy, type; } tmpcell;

static int cmp_tmpcell(const void* a, const void* b)
{
  const tmpcell* A = (const tmpcell*)a; const tmpcell* B = (const tmpcell*)b;
  return (A->key < B->key) ? -1 : (A->key > B->key) ? 1 : 0;
}

/* ------------------------------------------------------------- the builder */
typedef struct {
  int nx, ny;
  hmap split, solid, cell;    /* cell: (ix,iy) -> index into tmp[] (before sort) / storage index (after) */
  tmpcell* tmp; int64_t ntmp, captmp;
} blevel;

static int is_boundary_cell_kind(int kind)
{
  return kind == ORC_BC_DIRICHLET_EQ || kind == ORC_BC_DIRICHLET_EQ_RHO_EXTRAP || kind == ORC_BC_NEUMANN;
}

static int add_tmp(blevel* B, int ix, int iy, int type)
{
  if (B->ntmp == B->captmp) {
    int64_t nc = B->captmp ? 2 * B->captmp : 1024;
    tmpcell* t = (tmpcell*)realloc(B->tmp, (size_t)nc * sizeof(tmpcell));
    if (!t) return ORC_ENOMEM;
    B->tmp = t; B->captmp = nc;
  }
  tmpcell* c = &B->tmp[B->ntmp];
  c->ix = ix; c->iy = iy; c->type = type; c->key = 0;
  int rc = hmap_put(&B->cell, pack_xy(ix, iy), (int32_t)B->ntmp);
  if (rc) return rc;
  B->ntmp++;
  return ORC_OK;
}

/* periodic wrap of a target coordinate; returns 1 if inside the box afterwards */
static int wrap_axis(int* t, int n, int periodic)
{
  if (*t >= 0 && *t < n) return 1;
  if (!periodic) return 0;
  *t = ((*t % n) + n) % n;
  return 1;
}

int orc_build_levels(orc_grid* g, const int64_t* split_off, const int32_t* split_xy,
                     const int64_t* solid_off, const int32_t* solid_xy)
{
  const orc_config* cfg = &g->cfg;
  const int d = cfg->depth, Q = g->Q, W = g->W;
  const int perx = cfg->bc[0] == ORC_BC_PERIODIC, pery = cfg->bc[2] == ORC_BC_PERIODIC;
  if ((cfg->bc[0] == ORC_BC_PERIODIC) != (cfg->bc[1] == ORC_BC_PERIODIC)) return ORC_EINVAL;
  if ((cfg->bc[2] == ORC_BC_PERIODIC) != (cfg->bc[3] == ORC_BC_PERIODIC)) return ORC_EINVAL;
  if (d < 0 || d > 20 || cfg->nx_coarse < 1 || cfg->ny_coarse < 1) return ORC_EINVAL;
  int rc = ORC_OK;
  blevel* B = (blevel*)calloc((size_t)d + 1, sizeof(blevel));
  if (!B) return ORC_ENOMEM;

  /* split / solid sets */
  for (int l = 0; l <= d && !rc; ++l) {
    B[l].nx = cfg->nx_coarse << (d - l);
    B[l].ny = cfg->ny_coarse << (d - l);
    const int64_t ns = split_off ? split_off[l + 1] - split_off[l] : 0;
    const int64_t nz = solid_off ? solid_off[l + 1] - solid_off[l] : 0;
    if (l == 0 && ns != 0) { rc = ORC_EMESH; break; }
    if ((rc = hmap_init(&B[l].split, ns))) break;
    if ((rc = hmap_init(&B[l].solid, nz))) break;
    for (int64_t k = 0; k < ns; ++k) {
      const int ix = split_xy[2 * (split_off[l] + k)], iy = split_xy[2 * (split_off[l] + k) + 1];
      if (ix < 0 || iy < 0 || ix >= B[l].nx || iy >= B[l].ny) { rc = ORC_EMESH; break; }
      if ((rc = hmap_put(&B[l].split, pack_xy(ix, iy), 1))) break;
    }
    for (int64_t k = 0; k < nz && !rc; ++k) {
      const int ix = solid_xy[2 * (solid_off[l] + k)], iy = solid_xy[2 * (solid_off[l] + k) + 1];
      rc = hmap_put(&B[l].solid, pack_xy(ix, iy), 1);
    }
  }
  /* a split cell must exist: its parent is split (or it is on the coarsest level) and it is not solid */
  for (int l = 0; l < d && !rc; ++l)
    for (uint64_t p = 0; p < B[l].split.cap; ++p) {
      const uint64_t k = B[l].split.key[p];
      if (k == HKEY_EMPTY) continue;
      const int ix = (int)(uint32_t)(k >> 32) - CBIAS, iy = (int)(uint32_t)(k & 0xFFFFFFFFu) - CBIAS;
      if (hmap_get(&B[l + 1].split, pack_xy(ix >> 1, iy >> 1)) < 0) { rc = ORC_EMESH; break; }
    }

  /* top-down: leaves, coarse ghosts, fine ghosts */
  for (int l = d; l >= 0 && !rc; --l) {
    blevel* b = &B[l];
    int64_t expect = (l == d) ? (int64_t)b->nx * b->ny : 4 * B[l + 1].split.n + 4 * 1024;
    if ((rc = hmap_init(&b->cell, expect))) break;
    /* (1) leaves: cells that exist on this level, are not split and not solid */
    if (l == d) {
      for (int iy = 0; iy < b->ny && !rc; ++iy)
        for (int ix = 0; ix < b->nx && !rc; ++ix) {
          const uint64_t k = pack_xy(ix, iy);
          if (hmap_get(&b->split, k) >= 0 || hmap_get(&b->solid, k) >= 0) continue;
          rc = add_tmp(b, ix, iy, ORC_FLUID);
        }
    } else {
      const hmap* ps = &B[l + 1].split;
      for (uint64_t p = 0; p < ps->cap && !rc; ++p) {
        if (ps->key[p] == HKEY_EMPTY) continue;
        const int px = (int)(uint32_t)(ps->key[p] >> 32) - CBIAS, py = (int)(uint32_t)(ps->key[p] & 0xFFFFFFFFu) - CBIAS;
        for (int c = 0; c < 4 && !rc; ++c) {
          const int ix = 2 * px + (c & 1), iy = 2 * py + (c >> 1);
          const uint64_t k = pack_xy(ix, iy);
          if (hmap_get(&b->split, k) >= 0 || hmap_get(&b->solid, k) >= 0) continue;
          rc = add_tmp(b, ix, iy, ORC_FLUID);
        }
      }
      /* (3') fine ghosts handed down by level l+1 were appended below, after its own step (2) */
    }
    if (rc) break;
    /* fine ghosts: children of the coarse ghosts of level l+1, solid children not created */
    if (l < d) {
      blevel* c = &B[l + 1];
      for (int64_t t = 0; t < c->ntmp && !rc; ++t) {
        if (c->tmp[t].type != ORC_COARSE_GHOST) continue;
        for (int ch = 0; ch < 4 && !rc; ++ch) {
          const int ix = 2 * c->tmp[t].ix + (ch & 1), iy = 2 * c->tmp[t].iy + (ch >> 1);
          const uint64_t k = pack_xy(ix, iy);
          if (hmap_get(&b->solid, k) >= 0) continue;
          if (hmap_get(&b->cell, k) >= 0) { rc = ORC_EMESH; break; }
          rc = add_tmp(b, ix, iy, ORC_FINE_GHOST);
        }
      }
    }
    if (rc) break;
    /* (2) coarse ghost band: unsplit cells within Chebyshev distance W of a split cell (reading S4) */
    if (l >= 1) {
      for (uint64_t p = 0; p < b->split.cap && !rc; ++p) {
        if (b->split.key[p] == HKEY_EMPTY) continue;
        const int sx = (int)(uint32_t)(b->split.key[p] >> 32) - CBIAS, sy = (int)(uint32_t)(b->split.key[p] & 0xFFFFFFFFu) - CBIAS;
        for (int dy = -W; dy <= W && !rc; ++dy)
          for (int dx = -W; dx <= W; ++dx) {
            int tx = sx + dx, ty = sy + dy;
            if (!wrap_axis(&tx, b->nx, perx) || !wrap_axis(&ty, b->ny, pery)) continue;
            const int32_t t = hmap_get(&b->cell, pack_xy(tx, ty));
            if (t < 0) continue;     /* split, solid, or absent on this level (checked by the link validation) */
            if (b->tmp[t].type == ORC_FINE_GHOST) { rc = ORC_EMESH; break; }  /* interfaces too close */
            b->tmp[t].type = ORC_COARSE_GHOST;
          }
      }
    }
  }

  /* boundary cells, ordering, neighbour lists */
  for (int l = d; l >= 0 && !rc; --l) {
    blevel* b = &B[l];
    const int64_t n_inbox = b->ntmp;
    /* (5) boundary cells: W layers outside sides of kind DIRICHLET / NEUMANN */
    int anyb = 0;
    for (int s = 0; s < 4; ++s) anyb |= is_boundary_cell_kind(cfg->bc[s]);
    if (anyb) {
      for (int iy = -W; iy < b->ny + W && !rc; ++iy)
        for (int ix = -W; ix < b->nx + W && !rc; ++ix) {
          const int ox = ix < 0 ? 0 : (ix >= b->nx ? 1 : -1);
          const int oy = iy < 0 ? 2 : (iy >= b->ny ? 3 : -1);
          if (ox < 0 && oy < 0) { ix = b->nx - 1; continue; }   /* inside: jump to the right margin */
          if (ox >= 0 && !is_boundary_cell_kind(cfg->bc[ox])) continue;
          if (oy >= 0 && !is_boundary_cell_kind(cfg->bc[oy])) continue;
          const int cx = ix < 0 ? 0 : (ix >= b->nx ? b->nx - 1 : ix);
          const int cy = iy < 0 ? 0 : (iy >= b->ny ? b->ny - 1 : iy);
          const int32_t s = hmap_get(&b->cell, pack_xy(cx, cy));
          if (s < 0 || s >= n_inbox) continue;               /* source not stored on this level */
          if (b->tmp[s].type != ORC_FLUID) { rc = ORC_EMESH; break; }  /* interface touches the boundary */
          const int side = oy >= 0 ? oy : ox;
          const int kind = cfg->bc[side];
          rc = add_tmp(b, ix, iy, kind == ORC_BC_NEUMANN ? ORC_NEUMANN : ORC_DIRICHLET);
        }
    }
    if (rc) break;
    /* (6) order: in-box cells along the Z-curve, then boundary cells by (iy, ix) -- already generated in that order */
    for (int64_t t = 0; t < n_inbox; ++t) b->tmp[t].key = morton((uint32_t)b->tmp[t].ix, (uint32_t)b->tmp[t].iy);
    qsort(b->tmp, (size_t)n_inbox, sizeof(tmpcell), cmp_tmpcell);
    for (int64_t t = 0; t < b->ntmp; ++t) hmap_put(&b->cell, pack_xy(b->tmp[t].ix, b->tmp[t].iy), (int32_t)t);

    orc_level* L = &g->lv[l];
    L->n = b->ntmp; L->n_inbox = n_inbox;
    L->ix = (int32_t*)malloc(sizeof(int32_t) * (size_t)(L->n + 1));
    L->iy = (int32_t*)malloc(sizeof(int32_t) * (size_t)(L->n + 1));
    L->type = (int32_t*)malloc(sizeof(int32_t) * (size_t)(L->n + 1));
    L->aux = (int32_t*)malloc(sizeof(int32_t) * (size_t)(L->n + 1));
    L->nbr = (int32_t*)malloc(sizeof(int32_t) * (size_t)(L->n * (Q - 1) + 1));
    if (!L->ix || !L->iy || !L->type || !L->aux || !L->nbr) { rc = ORC_ENOMEM; break; }
    for (int64_t t = 0; t < L->n; ++t) {
      L->ix[t] = b->tmp[t].ix; L->iy[t] = b->tmp[t].iy; L->type[t] = b->tmp[t].type; L->aux[t] = -1;
    }
    /* (7) neighbour list: pull source of direction i is the cell at x - xi_i */
    for (int64_t t = 0; t < n_inbox && !rc; ++t) {
      for (int i = 1; i < Q; ++i) {
        int tx = L->ix[t] - orc_phys_cx(g->phys, i), ty = L->iy[t] - orc_phys_cy(g->phys, i);
        const int inx = wrap_axis(&tx, b->nx, perx), iny = wrap_axis(&ty, b->ny, pery);
        int32_t link;
        if (inx && iny) {
          const uint64_t k = pack_xy(tx, ty);
          const int32_t s = hmap_get(&b->cell, k);
          if (s >= 0) link = s;
          else if (hmap_get(&b->solid, k) >= 0) link = ORC_LINK_WALL;   /* bounce-back on solids */
          else link = ORC_LINK_NONE;
          if (link == ORC_LINK_NONE) {
            if (L->type[t] == ORC_FLUID) rc = ORC_EMESH;                          /* missing neighbour: no 2:1 band */
            if (L->type[t] == ORC_COARSE_GHOST && hmap_get(&b->split, k) < 0) rc = ORC_EMESH;
          }
        } else {
          const int ox = inx ? -1 : (tx < 0 ? 0 : 1);
          const int oy = iny ? -1 : (ty < 0 ? 2 : 3);
          const int prim = oy >= 0 ? oy : ox, sec = (oy >= 0 && ox >= 0) ? ox : -1;
          link = ORC_LINK_NONE;
          int side = prim;
          for (int pass = 0; pass < 2; ++pass) {
            const int kind = cfg->bc[side];
            if (kind == ORC_BC_WALL) { link = ORC_LINK_WALL; break; }
            if (kind == ORC_BC_MOVING_WALL || kind == ORC_BC_INFLOW_VBB) { link = ORC_LINK_VBB0 - side; break; }
            if (is_boundary_cell_kind(kind)) {
              const int32_t s = hmap_get(&b->cell, pack_xy(tx, ty));
              if (s >= 0) { link = s; break; }
            }
            if (sec < 0) break;
            side = sec;
          }
          if (link == ORC_LINK_NONE && L->type[t] != ORC_FINE_GHOST) rc = ORC_EMESH;
        }
        L->nbr[t * (Q - 1) + i - 1] = link;
      }
    }
    if (rc) break;
    /* boundary cells: NEUMANN replicates its source's row (reading S13); DIRICHLET has no links */
    for (int64_t t = n_inbox; t < L->n; ++t) {
      const int cx = L->ix[t] < 0 ? 0 : (L->ix[t] >= b->nx ? b->nx - 1 : L->ix[t]);
      const int cy = L->iy[t] < 0 ? 0 : (L->iy[t] >= b->ny ? b->ny - 1 : L->iy[t]);
      const int32_t s = hmap_get(&b->cell, pack_xy(cx, cy));
      L->aux[t] = s;
      for (int i = 1; i < Q; ++i)
        L->nbr[t * (Q - 1) + i - 1] = (L->type[t] == ORC_NEUMANN) ? L->nbr[(int64_t)s * (Q - 1) + i - 1] : ORC_LINK_NONE;
      if (L->type[t] == ORC_DIRICHLET) {
        /* remember the side in the ix/iy-independent way: encoded on demand by sim.c from ix, iy */
      }
    }
  }

  /* (8) ghost lists */
  for (int l = 1; l <= d && !rc; ++l) {
    orc_level* L = &g->lv[l];
    int64_t ng = 0;
    for (int64_t t = 0; t < L->n; ++t) ng += (L->type[t] == ORC_COARSE_GHOST);
    L->ng = ng;
    L->g_coarse = (int32_t*)malloc(sizeof(int32_t) * (size_t)(ng + 1));
    L->g_child = (int32_t*)malloc(sizeof(int32_t) * (size_t)(4 * ng + 1));
    L->g_mask = (uint64_t*)malloc(sizeof(uint64_t) * (size_t)(ng + 1));
    if (!L->g_coarse || !L->g_child || !L->g_mask) { rc = ORC_ENOMEM; break; }
    int64_t q = 0;
    for (int64_t t = 0; t < L->n; ++t) {
      if (L->type[t] != ORC_COARSE_GHOST) continue;
      L->aux[t] = (int32_t)q;
      L->g_coarse[q] = (int32_t)t;
      int nchild = 0;
      for (int ch = 0; ch < 4; ++ch) {
        const int32_t s = hmap_get(&B[l - 1].cell, pack_xy(2 * L->ix[t] + (ch & 1), 2 * L->iy[t] + (ch >> 1)));
        L->g_child[4 * q + ch] = s;
        nchild += (s >= 0);
      }
      uint64_t m = 0;
      for (int i = 1; i < Q; ++i)
        if (L->nbr[t * (Q - 1) + i - 1] == ORC_LINK_NONE) m |= (1ull << i);
      L->g_mask[q] = m;
      if (m && nchild == 0) rc = ORC_EMESH;
      ++q;
    }
  }

  for (int l = 0; l <= d; ++l) {
    hmap_free(&B[l].split); hmap_free(&B[l].solid); hmap_free(&B[l].cell);
    free(B[l].tmp);
  }
  free(B);
  return rc;
}
