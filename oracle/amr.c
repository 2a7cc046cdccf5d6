/* amr.c -- CPU ORACLE (test infrastructure, not the product): transfer of the state of one tree onto another when the
 * mesh is adapted (Sec. 8.1): "iterating over all cells in the updated tree and checking if corresponding LB
 * data exists at the same location in the previous tree.  If a match is found, populations are directly copied;
 * otherwise, they are recomputed using conservative coalescence (for cell coarsening) or uniform explosion (for cell
 * refinement)".
 *
 * Written as the definition, by recursion, cell by cell, with a linear search structure of its own (a sorted array per
 * level).  value(l, x, y) of the OLD tree:
 *   stored at (l, x, y)                           -> that state (copy);
 *   else, only for the cell asked for itself: the nearest stored ancestor (l+k, floor(x/2^k), floor(y/2^k))
 *                                                  -> that state (uniform explosion, Eq. 5, 7: all directions, lambda too);
 *   else                                           -> (1/N_f) sum over the N_f children (l-1, 2x+a, 2y+b) that have a
 *                                                     value (coalescence, Eq. 4, 6, all directions; solid children do
 *                                                     not exist), each evaluated by copy or coalescence.
 * A NEUMANN cell of the new tree takes the state its source cell received (it replicates that cell, S13).
 * Pins: tests/test_oracle_amr.py (identity on the same tree, exactness on uniform states, conservation of mass and
 * momentum to rounding, refine-then-coarsen returns the original values).                                            */
#include <stdlib.h>
#include <string.h>

#include "internal.h"

typedef struct { int64_t key; int32_t idx; } amr_ent;

static int64_t amr_key(int x, int y) { return ((int64_t)(y + (1 << 20)) << 32) | (int64_t)(x + (1 << 20)); }

static int amr_cmp(const void* a, const void* b)
{
  const int64_t ka = ((const amr_ent*)a)->key, kb = ((const amr_ent*)b)->key;
  return ka < kb ? -1 : ka > kb ? 1 : 0;
}

typedef struct { amr_ent* e; int64_t n; } amr_index;

static int32_t amr_find(const amr_index* ix, int x, int y)
{
  const int64_t k = amr_key(x, y);
  int64_t lo = 0, hi = ix->n - 1;
  while (lo <= hi) {
    const int64_t mid = (lo + hi) / 2;
    if (ix->e[mid].key == k) return ix->e[mid].idx;
    if (ix->e[mid].key < k) lo = mid + 1; else hi = mid - 1;
  }
  return -1;
}

static int floor_shift(int v, int k) { return v >= 0 ? v >> k : -((-v + (1 << k) - 1) >> k); }

/* copy or coalescence; returns 1 and fills out[npop] if the old tree has data for (l, x, y) */
static int amr_down(const orc_grid* src, const amr_index* ix, int l, int x, int y, double* out)
{
  const int np = src->npop;
  if (l <= src->depth) {
    const int32_t s = amr_find(&ix[l], x, y);
    if (s >= 0) {
      const orc_level* L = &src->lv[l];
      memcpy(out, L->S[L->cur] + (int64_t)s * np, sizeof(double) * (size_t)np);
      return 1;
    }
  }
  if (l == 0) return 0;
  double* sum = (double*)calloc((size_t)np, sizeof(double));
  double* ch = (double*)malloc(sizeof(double) * (size_t)np);
  int nf = 0;
  for (int k = 0; k < 4; ++k)
    if (amr_down(src, ix, l - 1, 2 * x + (k & 1), 2 * y + (k >> 1), ch)) {
      for (int p = 0; p < np; ++p) sum[p] += ch[p];
      ++nf;
    }
  for (int p = 0; p < np && nf > 0; ++p) out[p] = sum[p] / (double)nf;
  free(sum); free(ch);
  return nf > 0;
}

int orc_transfer(orc_grid* dst, const orc_grid* src)
{
  if (!dst || !src || dst->npop != src->npop || dst->Q != src->Q) return ORC_EINVAL;
  if (((int64_t)src->cfg.nx_coarse << src->depth) != ((int64_t)dst->cfg.nx_coarse << dst->depth) ||
      ((int64_t)src->cfg.ny_coarse << src->depth) != ((int64_t)dst->cfg.ny_coarse << dst->depth))
    return ORC_EINVAL;
  const int np = src->npop;
  amr_index* ix = (amr_index*)calloc((size_t)src->depth + 1, sizeof(amr_index));
  for (int l = 0; l <= src->depth; ++l) {
    const orc_level* L = &src->lv[l];
    ix[l].n = L->n;
    ix[l].e = (amr_ent*)malloc(sizeof(amr_ent) * (size_t)(L->n > 0 ? L->n : 1));
    for (int64_t c = 0; c < L->n; ++c) { ix[l].e[c].key = amr_key(L->ix[c], L->iy[c]); ix[l].e[c].idx = (int32_t)c; }
    qsort(ix[l].e, (size_t)L->n, sizeof(amr_ent), amr_cmp);
  }
  int rc = ORC_OK;
  for (int l = 0; l <= dst->depth && rc == ORC_OK; ++l) {
    orc_level* L = &dst->lv[l];
    L->cur = 0;
    for (int64_t c = 0; c < L->n && rc == ORC_OK; ++c) {
      double* out = L->S[0] + c * np;
      if (L->type[c] == ORC_NEUMANN) {             /* follows its source cell, stored before it */
        memcpy(out, L->S[0] + (int64_t)L->aux[c] * np, sizeof(double) * (size_t)np);
        continue;
      }
      const int x = L->ix[c], y = L->iy[c];
      int found = 0;
      if (l <= src->depth && amr_find(&ix[l], x, y) >= 0) found = amr_down(src, ix, l, x, y, out);
      for (int k = 1; !found && l + k <= src->depth; ++k) {
        const int32_t s = amr_find(&ix[l + k], floor_shift(x, k), floor_shift(y, k));
        if (s >= 0) {
          const orc_level* A = &src->lv[l + k];
          memcpy(out, A->S[A->cur] + (int64_t)s * np, sizeof(double) * (size_t)np);
          found = 1;
        }
      }
      if (!found) found = amr_down(src, ix, l, x, y, out);
      if (!found) rc = ORC_EMESH;
    }
    if (rc == ORC_OK) memcpy(L->S[1], L->S[0], sizeof(double) * (size_t)(L->n * np));
  }
  for (int l = 0; l <= src->depth; ++l) free(ix[l].e);
  free(ix);
  if (rc == ORC_OK) { dst->k = 0; dst->status = 0; }
  return rc;
}
