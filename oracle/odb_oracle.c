/*
 * odb_oracle.c -- CPU ORACLE for the ODB group -> align -> collate path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It
 * shares no code, header, table or helper with the CUDA path under
 * paper_2606_19989_b200/ and neither side imports the other.
 *
 * Plain, slow, sequential, single-threaded C.  Every routine follows the paper
 * (/root/reference/PAPER.md, cited as P:<line>) step by step, in the paper's order,
 * with the silent points fixed by the readings U1..U26 listed in DESIGN.md.
 * No blocking, fusion, closed forms or reordering: split is the literal while-loop of
 * Alg. 1, overflow is a literal sort, grouping is the literal threshold loop.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): App. D printed values, the
 * hand-worked examples E1..E6 (tests/golden/), closed forms for equal lengths,
 * declarative verifiers of the grouping / split / overflow rules, numpy.lexsort for the
 * sort, torch pad_sequence for collation, and the theorems' invariants (Lemma 1
 * partition, Lemma 2 potential, Thm 1 exactly-once, Thm 2 quota closure, Thm 4 bound).
 * Whole-pipeline parity against an external implementation: none exists ("parity
 * unpinned" beyond the pins above).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_RULE_THRESHOLD 0 /* paper section 2.2 */
#define ORACLE_RULE_MAXFIT_ASC 1 /* padded-area feasibility, App. I */
#define ORACLE_STOP_ALL_FINISHED 0
#define ORACLE_STOP_LOGICAL 1
#define ORACLE_STOP_QUOTA 2

/* ------------------------------------------------------------------------- */
/* small growable containers                                                 */
/* ------------------------------------------------------------------------- */
typedef struct {
    int32_t *v;
    int64_t n, cap;
} ivec;

static void ivec_push(ivec *a, int32_t x) {
    if (a->n == a->cap) {
        a->cap = a->cap ? a->cap * 2 : 16;
        a->v = (int32_t *)realloc(a->v, (size_t)a->cap * sizeof(int32_t));
    }
    a->v[a->n++] = x;
}

/* one candidate / emitted group: an ordered list of local sample ids (row order) */
typedef struct {
    int32_t *ids;
    int32_t n;
    int32_t orig; /* index of the candidate group (pre-alignment list) this group's samples came from */
} group;

typedef struct {
    group *g;
    int64_t n, cap;
} gvec;

static void gvec_insert(gvec *a, int64_t at, group x) {
    if (a->n == a->cap) {
        a->cap = a->cap ? a->cap * 2 : 16;
        a->g = (group *)realloc(a->g, (size_t)a->cap * sizeof(group));
    }
    memmove(a->g + at + 1, a->g + at, (size_t)(a->n - at) * sizeof(group));
    a->g[at] = x;
    a->n++;
}
static void gvec_push(gvec *a, group x) { gvec_insert(a, a->n, x); }

static group group_make(const int32_t *ids, int32_t n) {
    group g;
    g.n = n;
    g.orig = -1;
    g.ids = (int32_t *)malloc((size_t)(n > 0 ? n : 1) * sizeof(int32_t));
    if (n > 0) memcpy(g.ids, ids, (size_t)n * sizeof(int32_t));
    return g;
}

/* one emitted slot of a rank (a group, or an IDLE slot with count 0; reading U14) */
typedef struct {
    int32_t *ids;
    int32_t count;
    int32_t width;
    int32_t round;
    int32_t origin; /* step index of the first slot of this rank cut from the same candidate group */
} slot;

typedef struct {
    slot *s;
    int64_t n, cap;
} svec;

static void svec_push(svec *a, slot x) {
    if (a->n == a->cap) {
        a->cap = a->cap ? a->cap * 2 : 16;
        a->s = (slot *)realloc(a->s, (size_t)a->cap * sizeof(slot));
    }
    a->s[a->n++] = x;
}

/* ------------------------------------------------------------------------- */
/* sort: ascending by the composite key (len, sample_id)   (U1; section 2.2) */
/* ------------------------------------------------------------------------- */
static const int32_t *g_sort_len; /* lengths of the rank being sorted (single-threaded) */

static int cmp_len_id(const void *pa, const void *pb) {
    int32_t a = *(const int32_t *)pa, b = *(const int32_t *)pb;
    if (g_sort_len[a] != g_sort_len[b]) return g_sort_len[a] < g_sort_len[b] ? -1 : 1;
    return a < b ? -1 : (a > b ? 1 : 0);
}

/* Eq. 1 (floor confirmed at P:92; U11): B(l) = max(floor(L/l), 1) */
static int64_t target_group_size(int64_t budget, int64_t l) {
    int64_t b = budget / l;
    return b > 1 ? b : 1;
}
/* exposed so that the values App. D prints (B(800)=1, B(500)=2, B(100)=10) can be pinned */
int64_t oracle_target_group_size(int64_t budget, int64_t l) { return target_group_size(budget, l); }

/*
 * C.1 rule THRESHOLD -- section 2.2 P:36 and App. D, literally:
 *   sort ascending; iterate longest -> shortest with threshold t (initially 1);
 *   append to the current group; when its size reaches t finalise it and set
 *   t <- B(l) of the sample just added.  A partial tail group is emitted as is (U2).
 *   The list is then ordered short -> long with rows ascending (U3).
 * `order` = window ids already sorted ascending by (len,id).
 */
static void group_threshold(const int32_t *len, const int32_t *order, int32_t S, int64_t L, gvec *out) {
    gvec formed = {0, 0, 0}; /* in formation order (longest first) */
    int32_t *cur = (int32_t *)malloc((size_t)(S > 0 ? S : 1) * sizeof(int32_t));
    int32_t ncur = 0;
    int64_t t = 1;
    for (int32_t k = S - 1; k >= 0; --k) { /* longest -> shortest */
        int32_t id = order[k];
        cur[ncur++] = id;
        if (ncur >= t) {
            gvec_push(&formed, group_make(cur, ncur));
            t = target_group_size(L, len[id]);
            ncur = 0;
        }
    }
    if (ncur > 0) gvec_push(&formed, group_make(cur, ncur)); /* U2 */
    free(cur);
    /* U3: list short -> long; rows ascending = reverse each group, reverse the list */
    for (int64_t j = formed.n - 1; j >= 0; --j) {
        group g = formed.g[j];
        for (int32_t a = 0, b = g.n - 1; a < b; ++a, --b) {
            int32_t tmp = g.ids[a];
            g.ids[a] = g.ids[b];
            g.ids[b] = tmp;
        }
        gvec_push(out, g);
    }
    free(formed.g);
}

/*
 * C.2 rule MAXFIT_ASC -- App. I: feasibility on padded area,
 * max_i l_i * |b| <= budget, ascending greedy, singleton overflow allowed (U10).
 * Linear scan: extend while the extended group is still feasible.
 */
static void group_maxfit_asc(const int32_t *len, const int32_t *order, int32_t S, int64_t L, gvec *out) {
    int32_t i = 0;
    while (i < S) {
        int32_t e = i + 1;
        /* group order[i..e) ascending, so its max is len[order[e-1]]; try to add order[e] */
        while (e < S && (int64_t)(e + 1 - i) * (int64_t)len[order[e]] <= L) e++;
        gvec_push(out, group_make(order + i, e - i));
        i = e;
    }
}

/* ------------------------------------------------------------------------- */
/* Alg. 1: split and overflow on one rank's candidate list          */
/* ------------------------------------------------------------------------- */
/* Split (Alg.1 lines 3-6; U4, U5): while |G| < T: scanning from the last group
 * backward find the first group with >= 2 samples, extract its LAST sample (the longest,
 * rows are ascending) as a new singleton placed right after it. */
static void align_split(gvec *G, int64_t T) {
    while (G->n < T) {
        int64_t j = G->n - 1;
        while (j >= 0 && G->g[j].n < 2) j--;
        if (j < 0) break; /* no group with >= 2 samples (cannot happen when T <= S_r) */
        int32_t s = G->g[j].ids[G->g[j].n - 1];
        G->g[j].n -= 1;
        group single = group_make(&s, 1);
        single.orig = G->g[j].orig; /* the singleton still belongs to its candidate group (loss scaling, App. B) */
        gvec_insert(G, j + 1, single);
    }
}

typedef struct {
    int32_t count;
    int32_t index;
} cnt_idx;

static int cmp_count_desc_index_asc(const void *pa, const void *pb) {
    const cnt_idx *a = (const cnt_idx *)pa, *b = (const cnt_idx *)pb;
    if (a->count != b->count) return a->count > b->count ? -1 : 1;
    return a->index < b->index ? -1 : (a->index > b->index ? 1 : 0);
}

/* Overflow (Alg.1 line 8; U6, U7): sort groups by size (sample count) descending,
 * ties keep list order; keep the top T in that sorted order; the other groups' samples
 * go back to the buffer `back`. */
static void align_overflow(gvec *G, int64_t T, ivec *back) {
    int64_t n = G->n;
    cnt_idx *key = (cnt_idx *)malloc((size_t)n * sizeof(cnt_idx));
    for (int64_t j = 0; j < n; ++j) {
        key[j].count = G->g[j].n;
        key[j].index = (int32_t)j;
    }
    qsort(key, (size_t)n, sizeof(cnt_idx), cmp_count_desc_index_asc);
    group *kept = (group *)malloc((size_t)(T > 0 ? T : 1) * sizeof(group));
    for (int64_t j = 0; j < n; ++j) {
        group g = G->g[key[j].index];
        if (j < T) {
            kept[j] = g;
        } else {
            for (int32_t a = 0; a < g.n; ++a) ivec_push(back, g.ids[a]);
            free(g.ids);
        }
    }
    free(G->g);
    G->g = kept;
    G->n = T;
    G->cap = T > 0 ? T : 1;
    free(key);
}

/* ------------------------------------------------------------------------- */
/* the plan: everything except token movement                                  */
/* ------------------------------------------------------------------------- */
typedef struct {
    int32_t R;
    int64_t budget;
    int32_t rule, join_mode;
    int64_t sample_quota, emitted_so_far;
    int32_t buffer_size, slot_capacity;
    /* inputs (borrowed for the plan run only, copied here) */
    int64_t *rank_ptr;
    int32_t *lengths;
    /* results */
    int32_t n_rounds, n_steps, stop_reason;
    int64_t n_slots, total_elems, samples_emitted, samples_left, real_tokens, padded_elems;
    svec *slots; /* per rank */
    ivec *left;  /* per rank, ascending local ids */
    ivec round_T; /* T_grp of every emitting round */
    ivec step_samples;
    int64_t *grp_offset; /* n_slots, rank-major */
} oracle_plan;

static int cmp_i32(const void *pa, const void *pb) {
    int32_t a = *(const int32_t *)pa, b = *(const int32_t *)pb;
    return a < b ? -1 : (a > b ? 1 : 0);
}

/* exposed for direct pins of the grouping rules: groups one window.
 * ids[0..S) are local ids with lengths len[id]; outputs order[S] (rows of all groups
 * concatenated, list short->long) and gptr[G+1]; returns G. */
int64_t oracle_group_window(int32_t rule, int64_t budget, const int32_t *len, const int32_t *ids, int32_t S,
                            int32_t *order_out, int64_t *gptr_out) {
    int32_t *order = (int32_t *)malloc((size_t)(S > 0 ? S : 1) * sizeof(int32_t));
    memcpy(order, ids, (size_t)S * sizeof(int32_t));
    g_sort_len = len;
    qsort(order, (size_t)S, sizeof(int32_t), cmp_len_id);
    gvec G = {0, 0, 0};
    if (rule == ORACLE_RULE_THRESHOLD)
        group_threshold(len, order, S, budget, &G);
    else
        group_maxfit_asc(len, order, S, budget, &G);
    int64_t p = 0;
    gptr_out[0] = 0;
    for (int64_t j = 0; j < G.n; ++j) {
        for (int32_t a = 0; a < G.g[j].n; ++a) order_out[p++] = G.g[j].ids[a];
        gptr_out[j + 1] = p;
        free(G.g[j].ids);
    }
    int64_t n = G.n;
    free(G.g);
    free(order);
    return n;
}

/* exposed for direct pins of Alg. 1: align one rank's candidate list (given as CSR over
 * `rows`) to T groups.  Writes the aligned list (rows_out, gptr_out[T+1]) and the samples
 * returned to the buffer (back_out, *n_back).  Returns the aligned group count. */
int64_t oracle_align_list(const int32_t *rows, const int64_t *gptr, int64_t G, int64_t T, int32_t *rows_out,
                          int64_t *gptr_out, int32_t *back_out, int64_t *n_back) {
    gvec L = {0, 0, 0};
    for (int64_t j = 0; j < G; ++j) gvec_push(&L, group_make(rows + gptr[j], (int32_t)(gptr[j + 1] - gptr[j])));
    ivec back = {0, 0, 0};
    if (L.n < T)
        align_split(&L, T);
    else if (L.n > T)
        align_overflow(&L, T, &back);
    int64_t p = 0;
    gptr_out[0] = 0;
    for (int64_t j = 0; j < L.n; ++j) {
        for (int32_t a = 0; a < L.g[j].n; ++a) rows_out[p++] = L.g[j].ids[a];
        gptr_out[j + 1] = p;
        free(L.g[j].ids);
    }
    for (int64_t a = 0; a < back.n; ++a) back_out[a] = back.v[a];
    *n_back = back.n;
    int64_t n = L.n;
    free(L.g);
    free(back.v);
    return n;
}

/* Eq. 3 (Alg. 1 line 1; U8, U9, U23): exposed for pins.
 * G[r], S[r] per rank, C = slot capacity (0 = unlimited).  Active = G_r > 0. */
int64_t oracle_target_groups(const int64_t *G, const int64_t *S, int32_t R, int64_t C) {
    int64_t maxG = 0, cmin = -1, smin = -1; /* -1 = +infinity (empty positive minimum, U9) */
    for (int32_t r = 0; r < R; ++r) {
        if (G[r] <= 0) continue; /* not in A */
        if (G[r] > maxG) maxG = G[r];
        if (C > 0 && (cmin < 0 || C < cmin)) cmin = C;
        if (S[r] > 0 && (smin < 0 || S[r] < smin)) smin = S[r];
    }
    int64_t t = maxG;
    if (cmin >= 0 && cmin < t) t = cmin;
    if (smin >= 0 && smin < t) t = smin;
    return t > 1 ? t : 1;
}

void oracle_plan_free(oracle_plan *p) {
    if (!p) return;
    for (int32_t r = 0; r < p->R; ++r) {
        for (int64_t k = 0; k < p->slots[r].n; ++k) free(p->slots[r].s[k].ids);
        free(p->slots[r].s);
        free(p->left[r].v);
    }
    free(p->slots);
    free(p->left);
    free(p->round_T.v);
    free(p->step_samples.v);
    free(p->grp_offset);
    free(p->rank_ptr);
    free(p->lengths);
    free(p);
}

/*
 * C.3 the round loop (section 2.1; section 2.3; Alg. 1; App. C.1 with Q_r = {}).
 * Returns NULL with *err = 2 when some length < 1, *err = 1 on bad arguments.
 */
oracle_plan *oracle_plan_run_sched(int32_t R, int64_t budget, int32_t rule, int32_t join_mode, int64_t sample_quota,
                                   int64_t emitted_so_far, int32_t buffer_size, int32_t slot_capacity,
                                   const int32_t *lengths, const int64_t *rank_ptr, const int64_t *avail_sched,
                                   int32_t n_sched, int32_t *err);

oracle_plan *oracle_plan_run(int32_t R, int64_t budget, int32_t rule, int32_t join_mode, int64_t sample_quota,
                             int64_t emitted_so_far, int32_t buffer_size, int32_t slot_capacity,
                             const int32_t *lengths, const int64_t *rank_ptr, int32_t *err) {
    return oracle_plan_run_sched(R, budget, rule, join_mode, sample_quota, emitted_so_far, buffer_size, slot_capacity,
                                 lengths, rank_ptr, NULL, 0, err);
}

/*
 * The round loop with an ARRIVAL SCHEDULE (the asynchronous side of App. C.1: a sampler view sits in the
 * worker queue Q_r until the workers deliver it): in round j < n_sched only the first avail_sched[j*R + r]
 * views of rank r's stream have arrived and may be drained into B_r; from round n_sched on everything has.
 * A rank whose buffer is empty while views are still pending advertises n_groups = 0 ("insufficient data",
 * P:52), is not finished, and gets IDLE slots like any rank outside A; a round in which no rank has a group
 * is a SKIP round (no emission; Lemma 2: skip rounds are finite because the schedule is).
 */
oracle_plan *oracle_plan_run_sched(int32_t R, int64_t budget, int32_t rule, int32_t join_mode, int64_t sample_quota,
                                   int64_t emitted_so_far, int32_t buffer_size, int32_t slot_capacity,
                                   const int32_t *lengths, const int64_t *rank_ptr, const int64_t *avail_sched,
                                   int32_t n_sched, int32_t *err) {
    *err = 0;
    if (R < 1 || budget < 1 || (rule != 0 && rule != 1) || buffer_size < 0 || slot_capacity < 0) {
        *err = 1;
        return NULL;
    }
    int64_t N = rank_ptr[R];
    for (int64_t i = 0; i < N; ++i)
        if (lengths[i] < 1) {
            *err = 2;
            return NULL;
        }
    oracle_plan *p = (oracle_plan *)calloc(1, sizeof(oracle_plan));
    p->R = R;
    p->budget = budget;
    p->rule = rule;
    p->join_mode = join_mode;
    p->sample_quota = sample_quota;
    p->emitted_so_far = emitted_so_far;
    p->buffer_size = buffer_size;
    p->slot_capacity = slot_capacity;
    p->rank_ptr = (int64_t *)malloc((size_t)(R + 1) * sizeof(int64_t));
    memcpy(p->rank_ptr, rank_ptr, (size_t)(R + 1) * sizeof(int64_t));
    p->lengths = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
    memcpy(p->lengths, lengths, (size_t)N * sizeof(int32_t));
    p->slots = (svec *)calloc((size_t)R, sizeof(svec));
    p->left = (ivec *)calloc((size_t)R, sizeof(ivec));

    ivec *buf = (ivec *)calloc((size_t)R, sizeof(ivec));   /* B_r: collate buffer (ids) */
    int64_t *pos = (int64_t *)calloc((size_t)R, sizeof(int64_t)); /* next un-fetched view of R_r */
    gvec *cand = (gvec *)calloc((size_t)R, sizeof(gvec));
    int64_t *Gn = (int64_t *)calloc((size_t)R, sizeof(int64_t));
    int64_t *Sn = (int64_t *)calloc((size_t)R, sizeof(int64_t));
    int64_t s_emit = 0;
    int32_t round = 0;
    int stop = -1;

    while (stop < 0) {
        /* Fetch + Drain (App. C.1 P:299-303 with an empty worker queue): fill B_r up to buffer_size (U7, U8) */
        int32_t n_finished = 0;
        for (int32_t r = 0; r < R; ++r) {
            int64_t n_r = rank_ptr[r + 1] - rank_ptr[r];
            int64_t arrived = n_r; /* views of R_r the workers have delivered so far */
            if (avail_sched && round < n_sched && avail_sched[(int64_t)round * R + r] < n_r)
                arrived = avail_sched[(int64_t)round * R + r] > 0 ? avail_sched[(int64_t)round * R + r] : 0;
            while ((buffer_size == 0 || buf[r].n < buffer_size) && pos[r] < arrived) ivec_push(&buf[r], (int32_t)pos[r]++);
            Sn[r] = buf[r].n;
            /* status -1 "finished": nothing buffered and nothing pending; an empty buffer with views
             * still pending is status 0 "insufficient data" (unreachable without a schedule; U12) */
            if (Sn[r] == 0 && pos[r] == n_r) n_finished++;
        }
        /* termination predicates computed from the shared status (Thm 3 proof P:341) */
        if (join_mode && n_finished == R) {
            stop = ORACLE_STOP_ALL_FINISHED;
            round++;
            break;
        }
        if (!join_mode && n_finished > 0) {
            stop = ORACLE_STOP_LOGICAL;
            round++;
            break;
        }
        /* sort + greedy grouping per unfinished rank (section 2.2) */
        for (int32_t r = 0; r < R; ++r) {
            cand[r].n = 0;
            if (Sn[r] == 0) {
                Gn[r] = 0;
                continue;
            }
            const int32_t *len_r = lengths + rank_ptr[r];
            g_sort_len = len_r;
            qsort(buf[r].v, (size_t)buf[r].n, sizeof(int32_t), cmp_len_id);
            if (rule == ORACLE_RULE_THRESHOLD)
                group_threshold(len_r, buf[r].v, (int32_t)buf[r].n, budget, &cand[r]);
            else
                group_maxfit_asc(len_r, buf[r].v, (int32_t)buf[r].n, budget, &cand[r]);
            Gn[r] = cand[r].n; /* pre-alignment candidate count (U23) */
            for (int64_t j = 0; j < cand[r].n; ++j) cand[r].g[j].orig = (int32_t)j;
        }
        /* skip round: no rank produced a group (all "insufficient data" or finished): nothing is emitted */
        int any_active = 0;
        for (int32_t r = 0; r < R; ++r)
            if (Gn[r] > 0) any_active = 1;
        if (!any_active) {
            round++;
            continue;
        }
        /* Eq. 3 */
        int64_t T = oracle_target_groups(Gn, Sn, R, slot_capacity);
        ivec_push(&p->round_T, (int32_t)T);
        /* Alg. 1 per active rank; B_r <- returned samples (or empty) */
        for (int32_t r = 0; r < R; ++r) {
            if (Gn[r] == 0) continue;
            buf[r].n = 0;
            if (cand[r].n < T)
                align_split(&cand[r], T);
            else if (cand[r].n > T)
                align_overflow(&cand[r], T, &buf[r]);
        }
        /* emit step k = 0..T-1 (U26); finished ranks emit IDLE slots (U14) */
        int quota_hit = 0;
        int64_t k_emit = T;
        const int64_t step_base = p->step_samples.n; /* steps emitted by earlier rounds */
        for (int64_t k = 0; k < T; ++k) {
            int64_t e_k = 0;
            for (int32_t r = 0; r < R; ++r) {
                slot s;
                s.round = round;
                if (Gn[r] == 0) {
                    s.ids = (int32_t *)malloc(sizeof(int32_t));
                    s.count = 0;
                    s.width = 0;
                    s.origin = (int32_t)(step_base + k);
                } else {
                    group g = cand[r].g[k];
                    /* first aligned group cut from the same candidate: such groups are adjacent (a split
                     * singleton is inserted right after the group it came from, U5; groups kept by overflow
                     * are distinct candidates), so walk back over the run */
                    int64_t k0 = k;
                    while (k0 > 0 && cand[r].g[k0 - 1].orig == g.orig) k0--;
                    s.origin = (int32_t)(step_base + k0);
                    s.ids = g.ids; /* ownership moves to the slot */
                    s.count = g.n;
                    s.width = 0;
                    const int32_t *len_r = lengths + rank_ptr[r];
                    for (int32_t a = 0; a < g.n; ++a)
                        if (len_r[g.ids[a]] > s.width) s.width = len_r[g.ids[a]]; /* pad to group max (U18) */
                }
                svec_push(&p->slots[r], s);
                e_k += s.count;
            }
            ivec_push(&p->step_samples, (int32_t)e_k);
            s_emit += e_k;
            /* non-join sample-quota closure (Thm 2; U15): stop at the first step reaching Q */
            if (!join_mode && sample_quota > 0 && emitted_so_far + s_emit >= sample_quota) {
                quota_hit = 1;
                k_emit = k + 1;
                break;
            }
        }
        if (quota_hit) {
            /* groups k_emit.. of this round are not emitted: their samples stay in B_r */
            for (int32_t r = 0; r < R; ++r) {
                if (Gn[r] == 0) continue;
                for (int64_t k = k_emit; k < cand[r].n; ++k) {
                    for (int32_t a = 0; a < cand[r].g[k].n; ++a) ivec_push(&buf[r], cand[r].g[k].ids[a]);
                    free(cand[r].g[k].ids);
                }
            }
            stop = ORACLE_STOP_QUOTA;
        }
        round++;
    }

    p->n_rounds = round;
    p->stop_reason = stop;
    p->samples_emitted = s_emit;
    /* un-emitted views: B_r plus R_r (Lemma 1), ascending local id */
    for (int32_t r = 0; r < R; ++r) {
        int64_t n_r = rank_ptr[r + 1] - rank_ptr[r];
        for (int64_t a = 0; a < buf[r].n; ++a) ivec_push(&p->left[r], buf[r].v[a]);
        for (int64_t a = pos[r]; a < n_r; ++a) ivec_push(&p->left[r], (int32_t)a);
        qsort(p->left[r].v, (size_t)p->left[r].n, sizeof(int32_t), cmp_i32);
        p->samples_left += p->left[r].n;
    }
    /* every rank holds the same number of slots (U14) */
    p->n_steps = (int32_t)p->slots[0].n;
    for (int32_t r = 1; r < R; ++r)
        if (p->slots[r].n != p->n_steps) *err = 5;
    p->n_slots = (int64_t)R * p->n_steps;
    /* layout: rank-major slots, block offsets = exclusive scan of round_up(count*width, 16) */
    p->grp_offset = (int64_t *)malloc((size_t)(p->n_slots > 0 ? p->n_slots : 1) * sizeof(int64_t));
    int64_t off = 0;
    for (int32_t r = 0; r < R; ++r)
        for (int64_t k = 0; k < p->n_steps; ++k) {
            slot *s = &p->slots[r].s[k];
            int64_t area = (int64_t)s->count * (int64_t)s->width;
            p->grp_offset[(int64_t)r * p->n_steps + k] = off;
            off += (area + 15) / 16 * 16;
            p->padded_elems += area;
            for (int32_t a = 0; a < s->count; ++a) p->real_tokens += lengths[rank_ptr[r] + s->ids[a]];
        }
    p->total_elems = off;

    for (int32_t r = 0; r < R; ++r) {
        free(buf[r].v);
        free(cand[r].g);
    }
    free(buf);
    free(pos);
    free(cand);
    free(Gn);
    free(Sn);
    return p;
}

/* scalars: which = 0 n_rounds, 1 n_steps, 2 stop_reason, 3 n_slots, 4 total_elems, 5 samples_emitted,
 * 6 samples_left, 7 real_tokens, 8 padded_elems, 9 number of emitting rounds */
int64_t oracle_plan_scalar(const oracle_plan *p, int32_t which) {
    switch (which) {
    case 0: return p->n_rounds;
    case 1: return p->n_steps;
    case 2: return p->stop_reason;
    case 3: return p->n_slots;
    case 4: return p->total_elems;
    case 5: return p->samples_emitted;
    case 6: return p->samples_left;
    case 7: return p->real_tokens;
    case 8: return p->padded_elems;
    case 9: return p->round_T.n;
    default: return -1;
    }
}

/* tables; any pointer may be NULL.  Sizes: per-slot arrays n_slots; grp_sample_ptr n_slots+1;
 * grp_sample_ids samples_emitted; step_samples n_steps; left_ptr R+1; left_ids samples_left;
 * round_T (number of emitting rounds). */
void oracle_plan_tables(const oracle_plan *p, int32_t *grp_count, int32_t *grp_width, int32_t *grp_round,
                        int64_t *grp_offset, int32_t *grp_real_tokens, int64_t *grp_sample_ptr,
                        int32_t *grp_sample_ids, int32_t *step_samples, int64_t *left_ptr, int32_t *left_ids,
                        int32_t *round_T) {
    int64_t q = 0;
    for (int32_t r = 0; r < p->R; ++r)
        for (int64_t k = 0; k < p->n_steps; ++k) {
            int64_t s = (int64_t)r * p->n_steps + k;
            const slot *sl = &p->slots[r].s[k];
            if (grp_count) grp_count[s] = sl->count;
            if (grp_width) grp_width[s] = sl->width;
            if (grp_round) grp_round[s] = sl->round;
            if (grp_offset) grp_offset[s] = p->grp_offset[s];
            if (grp_real_tokens) {
                int64_t t = 0;
                for (int32_t a = 0; a < sl->count; ++a) t += p->lengths[p->rank_ptr[r] + sl->ids[a]];
                grp_real_tokens[s] = (int32_t)t;
            }
            if (grp_sample_ptr) grp_sample_ptr[s] = q;
            for (int32_t a = 0; a < sl->count; ++a) {
                if (grp_sample_ids) grp_sample_ids[q] = sl->ids[a];
                q++;
            }
        }
    if (grp_sample_ptr) grp_sample_ptr[p->n_slots] = q;
    if (step_samples)
        for (int64_t k = 0; k < p->n_steps; ++k) step_samples[k] = p->step_samples.v[k];
    int64_t lq = 0;
    for (int32_t r = 0; r < p->R; ++r) {
        if (left_ptr) left_ptr[r] = lq;
        for (int64_t a = 0; a < p->left[r].n; ++a) {
            if (left_ids) left_ids[lq] = p->left[r].v[a];
            lq++;
        }
    }
    if (left_ptr) left_ptr[p->R] = lq;
    if (round_T)
        for (int64_t a = 0; a < p->round_T.n; ++a) round_T[a] = p->round_T.v[a];
}

/* per-slot origin (n_slots, rank-major): see `slot.origin` */
void oracle_plan_origin(const oracle_plan *p, int32_t *grp_origin) {
    for (int32_t r = 0; r < p->R; ++r)
        for (int64_t k = 0; k < p->n_steps; ++k) grp_origin[(int64_t)r * p->n_steps + k] = p->slots[r].s[k].origin;
}

/*
 * Loss-scaling weights w_{r,k} per slot (rank-major [R][n_steps]), fp64; DDP prescales rank r's mean loss
 * of step k by W * w_{r,k} (section 2.3 "Loss scaling" P:60-65; App. B; the three modes P:738).
 *   mode 1 sample-level:        w = n_{r,k} / N_k,           N_k = sum_r n_{r,k}            (P:65, P:738 (1))
 *   mode 3 exact token-level:   w = t_{r,k} / T_tok,k,       T_tok,k = sum_r t_{r,k}        (Eq. 2)
 *          with t = the POST-alignment valid-token count of the slot.
 *   mode 2 approximate token-level: t_adj = n_adj * tbar, tbar = t_orig / n_orig of the PRE-alignment
 *          candidate group the slot was cut from (P:283, P:738 (2); reading U27); w = t_adj / sum_r t_adj.
 * A step whose denominator is 0 gets weight 0 on every rank.  Sums run over ranks in the order r = 0..R-1.
 * count/valid/origin: the per-slot tables (origin = step index of the first slot cut from the same candidate).
 */
void oracle_loss_weights(int32_t mode, int32_t R, int64_t n_steps, const int32_t *count, const int32_t *valid,
                         const int32_t *origin, double *w) {
    for (int64_t k = 0; k < n_steps; ++k) {
        double denom = 0.0;
        for (int32_t r = 0; r < R; ++r) {
            int64_t s = (int64_t)r * n_steps + k;
            double num;
            if (mode == 1) {
                num = (double)count[s];
            } else if (mode == 3) {
                num = (double)valid[s];
            } else {
                int64_t t_orig = 0, n_orig = 0;
                for (int64_t k2 = 0; k2 < n_steps; ++k2) { /* every slot of this rank cut from the same candidate */
                    int64_t s2 = (int64_t)r * n_steps + k2;
                    if (origin[s2] == origin[s]) {
                        t_orig += valid[s2];
                        n_orig += count[s2];
                    }
                }
                double tbar = n_orig > 0 ? (double)t_orig / (double)n_orig : 0.0;
                num = (double)count[s] * tbar;
            }
            w[s] = num;
            denom = denom + num;
        }
        for (int32_t r = 0; r < R; ++r) {
            int64_t s = (int64_t)r * n_steps + k;
            w[s] = denom > 0.0 ? w[s] / denom : 0.0;
        }
    }
}

/* is token position t of a sample inside one of its masked spans [lo,hi)?  linear scan */
static int masked_at(int64_t t, const int32_t *lo, const int32_t *hi, int64_t nspan) {
    for (int64_t j = 0; j < nspan; ++j)
        if (t >= lo[j] && t < hi[j]) return 1;
    return 0;
}

/*
 * C.4 collation of one slot (collate_fn P:28; pad to the group max P:416-420; tensor
 * contract from BASELINE.json north_star; U16, U17, U18).  Dense [count x width],
 * right-padded.  tok_start[g] = offset of global sample g's first token in `tokens`
 * (only the slot's samples are dereferenced).  Outputs are count*width elements each.
 * Returns the slot's valid-token count = #{labels != ignore_index} (Eq. 2).
 */
int64_t oracle_collate_slot(const oracle_plan *p, int64_t slot_index, const int32_t *tokens,
                            const int64_t *tok_start, const int64_t *span_ptr, const int32_t *span_lo,
                            const int32_t *span_hi, int32_t pad_id, int32_t ignore_index, int32_t shift_labels,
                            int32_t *input_ids, uint8_t *attention_mask, int32_t *position_ids, int32_t *labels) {
    int32_t r = (int32_t)(slot_index / (p->n_steps > 0 ? p->n_steps : 1));
    int64_t k = slot_index - (int64_t)r * p->n_steps;
    const slot *sl = &p->slots[r].s[k];
    int64_t width = sl->width, valid = 0;
    for (int32_t b = 0; b < sl->count; ++b) {
        int64_t g = p->rank_ptr[r] + sl->ids[b];
        int64_t len_b = p->lengths[g];
        const int32_t *tok = tokens + tok_start[g];
        const int32_t *lo = span_lo + span_ptr[g];
        const int32_t *hi = span_hi + span_ptr[g];
        int64_t nspan = span_ptr[g + 1] - span_ptr[g];
        for (int64_t t = 0; t < width; ++t) {
            int64_t o = (int64_t)b * width + t;
            int real = t < len_b;
            int32_t lab;
            if (shift_labels)
                lab = (t + 1 < len_b && !masked_at(t + 1, lo, hi, nspan)) ? tok[t + 1] : ignore_index;
            else
                lab = (real && !masked_at(t, lo, hi, nspan)) ? tok[t] : ignore_index;
            if (input_ids) input_ids[o] = real ? tok[t] : pad_id;
            if (attention_mask) attention_mask[o] = real ? 1 : 0;
            if (position_ids) position_ids[o] = real ? (int32_t)t : 0;
            if (labels) labels[o] = lab;
            if (lab != ignore_index) valid++;
        }
    }
    return valid;
}

/* all slots into the four flat arenas at grp_offset (gap elements are never written);
 * grp_valid_tokens[n_slots], step_valid_tokens[n_steps] (sum over ranks; Eq. 2). */
void oracle_collate_all(const oracle_plan *p, const int32_t *tokens, const int64_t *tok_start,
                        const int64_t *span_ptr, const int32_t *span_lo, const int32_t *span_hi, int32_t pad_id,
                        int32_t ignore_index, int32_t shift_labels, int32_t *input_ids, uint8_t *attention_mask,
                        int32_t *position_ids, int32_t *labels, int32_t *grp_valid_tokens,
                        int64_t *step_valid_tokens) {
    for (int64_t k = 0; k < p->n_steps; ++k)
        if (step_valid_tokens) step_valid_tokens[k] = 0;
    for (int64_t s = 0; s < p->n_slots; ++s) {
        int64_t off = p->grp_offset[s];
        int64_t v = oracle_collate_slot(p, s, tokens, tok_start, span_ptr, span_lo, span_hi, pad_id, ignore_index,
                                        shift_labels, input_ids ? input_ids + off : NULL,
                                        attention_mask ? attention_mask + off : NULL,
                                        position_ids ? position_ids + off : NULL, labels ? labels + off : NULL);
        if (grp_valid_tokens) grp_valid_tokens[s] = (int32_t)v;
        if (step_valid_tokens) step_valid_tokens[s % (p->n_steps > 0 ? p->n_steps : 1)] += v;
    }
}

/* The loop of oracle_collate_all restricted to the slots [slot_lo, slot_hi) (one rank's slots, say),
 * written into buffers whose element 0 is arena element elem_base: the full-size parity tests compare
 * rank by rank so that neither side holds 28 GB on the host.  No arithmetic of its own: every element
 * comes from oracle_collate_slot.  grp_valid_tokens: slot_hi - slot_lo entries. */
void oracle_collate_range(const oracle_plan *p, int64_t slot_lo, int64_t slot_hi, int64_t elem_base,
                          const int32_t *tokens, const int64_t *tok_start, const int64_t *span_ptr,
                          const int32_t *span_lo, const int32_t *span_hi, int32_t pad_id, int32_t ignore_index,
                          int32_t shift_labels, int32_t *input_ids, uint8_t *attention_mask, int32_t *position_ids,
                          int32_t *labels, int32_t *grp_valid_tokens) {
    for (int64_t s = slot_lo; s < slot_hi; ++s) {
        int64_t off = p->grp_offset[s] - elem_base;
        int64_t v = oracle_collate_slot(p, s, tokens, tok_start, span_ptr, span_lo, span_hi, pad_id, ignore_index,
                                        shift_labels, input_ids ? input_ids + off : NULL,
                                        attention_mask ? attention_mask + off : NULL,
                                        position_ids ? position_ids + off : NULL, labels ? labels + off : NULL);
        if (grp_valid_tokens) grp_valid_tokens[s - slot_lo] = (int32_t)v;
    }
}

/* ========================================================================================= */
/* the paper's OFFLINE comparators as planners (App. I; App. J).
 * They see a GLOBAL scalar length array (the "oracle cache"), build one global batch list that every rank
 * computes identically, and hand batches to the W ranks by striding; a slot's ids are therefore GLOBAL
 * sample ids (the plan's rank_ptr is all zeros).  Random numbers are inputs: `perm` (the epoch-seeded
 * shuffle, a permutation of 0..N-1) and `shuffle_key` (one non-negative key per potential batch index; the
 * batch shuffle orders batches by (key, index)).
 *
 *   GMT (planner 0): "ascending-length sort plus greedy packing against a max-token budget", feasibility on
 *       padded area max_i l_i * |b| <= budget, "singleton overflows allowed".
 *   BMT (planner 1): "epoch-seeded shuffle, sample-count buckets, within-bucket length sort, greedy packing,
 *       then batch shuffle".  Readings (U30): a bucket = `size` consecutive entries of the
 *       shuffled order (the last one ragged); the within-bucket sort is ascending by (length, position in the
 *       shuffled order); packing never crosses a bucket boundary.
 *   both: "The list is then padded to a multiple of the world size by wrap-around repetition of the leading
 *       batches and assigned to ranks by striding": G batches -> n_steps = ceil(G / W), slot (r, k) =
 *       batch (k W + r) mod G.
 *   HFG (planner 2): "samples a random permutation, partitions it into megabatches, sorts each megabatch by the
 *       oracle post-tokenization length, concatenates the megabatches, pads the index list to a multiple of
 *       world size, and stride-shards it across ranks ... keeps a fixed batch size".  Readings (U31):
 *       the megabatch sort is DESCENDING (the HuggingFace group_by_length convention the paper names), ties by
 *       descending position in the permutation (= the reverse of the ascending (length, position) order);
 *       padding repeats the leading indices; rank r's list is every W-th index from r; its steps are runs of
 *       `batch_size` consecutive entries (the last one ragged), rows in list order.
 * Slot width = the longest sample of the slot (pad to max).  round = 0, origin = own step,
 * stop_reason = ALL_FINISHED, n_rounds = 1. */
static void offline_finish(oracle_plan *p, int32_t *err) {
    int32_t R = p->R;
    p->n_steps = (int32_t)p->slots[0].n;
    for (int32_t r = 1; r < R; ++r)
        if (p->slots[r].n != p->n_steps) *err = 5;
    p->n_slots = (int64_t)R * p->n_steps;
    p->grp_offset = (int64_t *)malloc((size_t)(p->n_slots > 0 ? p->n_slots : 1) * sizeof(int64_t));
    int64_t off = 0;
    for (int32_t r = 0; r < R; ++r)
        for (int64_t k = 0; k < p->n_steps; ++k) {
            slot *s = &p->slots[r].s[k];
            s->width = 0;
            for (int32_t a = 0; a < s->count; ++a)
                if (p->lengths[s->ids[a]] > s->width) s->width = p->lengths[s->ids[a]];
            int64_t area = (int64_t)s->count * (int64_t)s->width;
            p->grp_offset[(int64_t)r * p->n_steps + k] = off;
            off += (area + 15) / 16 * 16;
            p->padded_elems += area;
            p->samples_emitted += s->count;
            for (int32_t a = 0; a < s->count; ++a) p->real_tokens += p->lengths[s->ids[a]];
        }
    p->total_elems = off;
    for (int64_t k = 0; k < p->n_steps; ++k) {
        int64_t e = 0;
        for (int32_t r = 0; r < R; ++r) e += p->slots[r].s[k].count;
        ivec_push(&p->step_samples, (int32_t)e);
    }
    p->n_rounds = 1;
    p->stop_reason = ORACLE_STOP_ALL_FINISHED;
}

static const int32_t *g_key_ptr; /* batch shuffle keys (single-threaded) */
static int cmp_key_index(const void *pa, const void *pb) {
    int32_t a = *(const int32_t *)pa, b = *(const int32_t *)pb;
    if (g_key_ptr[a] != g_key_ptr[b]) return g_key_ptr[a] < g_key_ptr[b] ? -1 : 1;
    return a < b ? -1 : (a > b ? 1 : 0);
}

oracle_plan *oracle_offline_plan(int32_t planner, int32_t W, int64_t budget, const int32_t *len, int64_t N,
                                 const int32_t *perm, const int32_t *shuffle_key, int32_t size, int32_t batch_size,
                                 int32_t *err) {
    *err = 0;
    if (W < 1 || N < 0 || planner < 0 || planner > 2 || (planner != 0 && !perm && N > 0) ||
        (planner == 1 && (!shuffle_key || size < 1)) || (planner == 2 && (size < 1 || batch_size < 1)) ||
        (planner != 2 && budget < 1)) {
        *err = 1;
        return NULL;
    }
    for (int64_t i = 0; i < N; ++i)
        if (len[i] < 1) {
            *err = 2;
            return NULL;
        }
    oracle_plan *p = (oracle_plan *)calloc(1, sizeof(oracle_plan));
    p->R = W;
    p->budget = budget;
    p->rule = ORACLE_RULE_MAXFIT_ASC;
    p->join_mode = 1;
    p->rank_ptr = (int64_t *)calloc((size_t)W + 1, sizeof(int64_t)); /* all zeros: slot ids are global ids */
    p->lengths = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
    if (N > 0) memcpy(p->lengths, len, (size_t)N * sizeof(int32_t));
    p->slots = (svec *)calloc((size_t)W, sizeof(svec));
    p->left = (ivec *)calloc((size_t)W, sizeof(ivec));
    if (planner == 2) {
        /* HFG: per-megabatch descending sort of the permutation, concatenated */
        int32_t *L = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
        int32_t *plen = (int32_t *)malloc((size_t)(size > 0 ? size : 1) * sizeof(int32_t));
        int32_t *loc = (int32_t *)malloc((size_t)(size > 0 ? size : 1) * sizeof(int32_t));
        for (int64_t m0 = 0; m0 < N; m0 += size) {
            int32_t n = (int32_t)((N - m0 < size) ? (N - m0) : size);
            for (int32_t a = 0; a < n; ++a) {
                plen[a] = len[perm[m0 + a]];
                loc[a] = a;
            }
            g_sort_len = plen;
            qsort(loc, (size_t)n, sizeof(int32_t), cmp_len_id); /* ascending (length, position) ... */
            for (int32_t a = 0; a < n; ++a) L[m0 + a] = perm[m0 + loc[n - 1 - a]]; /* ... read backwards */
        }
        int64_t n_per = (N + W - 1) / W; /* the index list padded to a multiple of W, one stride per rank */
        for (int32_t r = 0; r < W; ++r)
            for (int64_t i0 = 0; i0 < n_per; i0 += batch_size) {
                int64_t n = (n_per - i0 < batch_size) ? (n_per - i0) : batch_size;
                slot s;
                memset(&s, 0, sizeof(s));
                s.ids = (int32_t *)malloc((size_t)n * sizeof(int32_t));
                s.count = (int32_t)n;
                s.origin = (int32_t)(i0 / batch_size);
                for (int64_t a = 0; a < n; ++a) s.ids[a] = L[((i0 + a) * W + r) % N]; /* wrap-around padding */
                svec_push(&p->slots[r], s);
            }
        free(L);
        free(plen);
        free(loc);
    } else {
        gvec batches;
        memset(&batches, 0, sizeof(batches));
        if (planner == 0) {
            int32_t *order = (int32_t *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int32_t));
            for (int64_t i = 0; i < N; ++i) order[i] = (int32_t)i;
            g_sort_len = len;
            qsort(order, (size_t)N, sizeof(int32_t), cmp_len_id);
            group_maxfit_asc(len, order, (int32_t)N, budget, &batches);
            free(order);
        } else {
            int32_t *plen = (int32_t *)malloc((size_t)size * sizeof(int32_t));
            int32_t *loc = (int32_t *)malloc((size_t)size * sizeof(int32_t));
            int32_t *ord = (int32_t *)malloc((size_t)size * sizeof(int32_t));
            gvec pre;
            memset(&pre, 0, sizeof(pre));
            for (int64_t b0 = 0; b0 < N; b0 += size) {
                int32_t n = (int32_t)((N - b0 < size) ? (N - b0) : size);
                for (int32_t a = 0; a < n; ++a) {
                    plen[a] = len[perm[b0 + a]];
                    loc[a] = a;
                }
                g_sort_len = plen;
                qsort(loc, (size_t)n, sizeof(int32_t), cmp_len_id);
                for (int32_t a = 0; a < n; ++a) ord[a] = perm[b0 + loc[a]];
                group_maxfit_asc(len, ord, n, budget, &pre); /* packing never leaves the bucket */
            }
            /* batch shuffle: order by (key, index) */
            int32_t *idx = (int32_t *)malloc((size_t)(pre.n > 0 ? pre.n : 1) * sizeof(int32_t));
            for (int64_t j = 0; j < pre.n; ++j) idx[j] = (int32_t)j;
            g_key_ptr = shuffle_key;
            qsort(idx, (size_t)pre.n, sizeof(int32_t), cmp_key_index);
            for (int64_t j = 0; j < pre.n; ++j) gvec_push(&batches, pre.g[idx[j]]);
            free(idx);
            free(pre.g);
            free(plen);
            free(loc);
            free(ord);
        }
        /* wrap-around repetition of the leading batches to a multiple of W, then striding */
        int64_t G = batches.n, n_steps = (G + W - 1) / W;
        for (int32_t r = 0; r < W; ++r)
            for (int64_t k = 0; k < n_steps; ++k) {
                const group *g = &batches.g[(k * W + r) % G];
                slot s;
                memset(&s, 0, sizeof(s));
                s.ids = (int32_t *)malloc((size_t)(g->n > 0 ? g->n : 1) * sizeof(int32_t));
                memcpy(s.ids, g->ids, (size_t)g->n * sizeof(int32_t));
                s.count = g->n;
                s.origin = (int32_t)k;
                svec_push(&p->slots[r], s);
            }
        for (int64_t j = 0; j < G; ++j) free(batches.g[j].ids);
        free(batches.g);
    }
    offline_finish(p, err);
    return p;
}
