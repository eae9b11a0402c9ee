/*
 * workload_routing.c -- host-side shortest-route generator for the SYNTHETIC benchmark inputs.
 *
 * Routing is outside the timed path ("excluding routing and initialisation"; the paper
 * runs a priority-queue Dijkstra on CPUs).  This file only manufactures inputs for
 * manta_load_trips: for every (origin node, destination node) pair it returns the edge sequence of a
 * shortest path under the given non-negative edge weights.  It holds none of the simulator's
 * arithmetic and is used by the tests (to feed oracle AND CUDA path the same routes) and by bench.py.
 *
 * Method: trips are grouped by origin; one binary-heap Dijkstra per distinct origin, stopped as soon
 * as every destination of that origin is settled; pthreads pull origins from a shared counter.
 * Deterministic: a node's parent edge is the first edge that reaches its final distance under
 * strict '<' relaxation with the heap ordered by (distance, node id), independent of thread count.
 */
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct { double d; uint32_t u; } hent;

typedef struct {
    uint32_t n_nodes;
    const uint32_t *row_ptr, *head;
    const double *w;
    uint32_t n_groups;
    const uint32_t *grp_ptr;   /* [n_groups+1] into sorted trip list */
    const uint32_t *trip_sorted; /* trip indices sorted by origin */
    const uint32_t *origin, *dest;
    uint32_t *route_len;       /* [n_trips] out */
    uint32_t **route_buf;      /* [n_trips] out: malloc'd edge list per trip (reversed order fixed) */
    volatile uint32_t next;
    pthread_mutex_t mu;
    int failed;
} job;

static void heap_push(hent *h, uint32_t *n, hent x)
{
    uint32_t i = (*n)++;
    while (i > 0) {
        uint32_t p = (i - 1) >> 1;
        if (h[p].d < x.d || (h[p].d == x.d && h[p].u <= x.u)) break;
        h[i] = h[p];
        i = p;
    }
    h[i] = x;
}
static hent heap_pop(hent *h, uint32_t *n)
{
    hent top = h[0], x = h[--(*n)];
    uint32_t i = 0, m = *n;
    for (;;) {
        uint32_t c = 2 * i + 1;
        if (c >= m) break;
        if (c + 1 < m && (h[c + 1].d < h[c].d || (h[c + 1].d == h[c].d && h[c + 1].u < h[c].u))) c++;
        if (x.d < h[c].d || (x.d == h[c].d && x.u <= h[c].u)) break;
        h[i] = h[c];
        i = c;
    }
    h[i] = x;
    return top;
}

static void *worker(void *arg)
{
    job *J = (job *)arg;
    uint32_t n = J->n_nodes;
    double *dist = (double *)malloc(sizeof(double) * n);
    uint32_t *par = (uint32_t *)malloc(sizeof(uint32_t) * n);   /* parent EDGE */
    uint32_t *stamp = (uint32_t *)calloc(n, sizeof(uint32_t));  /* visit epoch */
    uint8_t *want = (uint8_t *)calloc(n, 1);
    uint8_t *done = (uint8_t *)calloc(n, 1);
    uint32_t *touched = (uint32_t *)malloc(sizeof(uint32_t) * n);
    uint32_t m_edges = J->row_ptr[n];
    hent *heap = (hent *)malloc(sizeof(hent) * ((size_t)m_edges + n + 16));
    uint32_t *tail_of = NULL;
    uint32_t epoch = 0;
    /* tail node of each edge, needed to walk parents back */
    tail_of = (uint32_t *)malloc(sizeof(uint32_t) * (m_edges + 1));
    for (uint32_t u = 0; u < n; u++)
        for (uint32_t e = J->row_ptr[u]; e < J->row_ptr[u + 1]; e++) tail_of[e] = u;
    for (;;) {
        pthread_mutex_lock(&J->mu);
        uint32_t g = J->next++;
        pthread_mutex_unlock(&J->mu);
        if (g >= J->n_groups) break;
        uint32_t b = J->grp_ptr[g], e_ = J->grp_ptr[g + 1];
        uint32_t src = J->origin[J->trip_sorted[b]];
        uint32_t remaining = 0, n_touched = 0, hn = 0;
        epoch++;
        for (uint32_t k = b; k < e_; k++) {
            uint32_t d = J->dest[J->trip_sorted[k]];
            if (!want[d]) { want[d] = 1; remaining++; }
        }
        dist[src] = 0.0; stamp[src] = epoch; par[src] = 0xFFFFFFFFu; touched[n_touched++] = src;
        heap_push(heap, &hn, (hent){0.0, src});
        while (hn > 0 && remaining > 0) {
            hent x = heap_pop(heap, &hn);
            uint32_t u = x.u;
            if (done[u] || x.d > dist[u]) continue;
            done[u] = 1;
            if (want[u]) { want[u] = 2; remaining--; }
            for (uint32_t e = J->row_ptr[u]; e < J->row_ptr[u + 1]; e++) {
                uint32_t v = J->head[e];
                double nd = x.d + J->w[e];
                if (stamp[v] != epoch) {
                    stamp[v] = epoch; dist[v] = nd; par[v] = e; touched[n_touched++] = v;
                    heap_push(heap, &hn, (hent){nd, v});
                } else if (!done[v] && nd < dist[v]) {
                    dist[v] = nd; par[v] = e;
                    heap_push(heap, &hn, (hent){nd, v});
                }
            }
        }
        for (uint32_t k = b; k < e_; k++) {
            uint32_t tr = J->trip_sorted[k];
            uint32_t d = J->dest[tr];
            if (stamp[d] != epoch || !done[d] || d == src) { /* unreachable or empty */
                J->route_len[tr] = 0; J->route_buf[tr] = NULL;
                if (d != src) J->failed = 1;
                continue;
            }
            uint32_t len = 0;
            for (uint32_t v = d; v != src; v = tail_of[par[v]]) len++;
            uint32_t *r = (uint32_t *)malloc(sizeof(uint32_t) * len);
            uint32_t i = len;
            for (uint32_t v = d; v != src; v = tail_of[par[v]]) r[--i] = par[v];
            J->route_len[tr] = len;
            J->route_buf[tr] = r;
        }
        for (uint32_t k = 0; k < n_touched; k++) { done[touched[k]] = 0; }
        for (uint32_t k = b; k < e_; k++) want[J->dest[J->trip_sorted[k]]] = 0;
    }
    free(dist); free(par); free(stamp); free(want); free(done); free(touched); free(heap); free(tail_of);
    return NULL;
}

typedef struct { uint32_t key, idx; } ki;
static int cmp_ki(const void *a, const void *b)
{
    const ki *x = (const ki *)a, *y = (const ki *)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return x->idx < y->idx ? -1 : (x->idx > y->idx);
}

/* Returns 0 on success, 1 if some destination was unreachable (its route is left empty).
 * *out_route_edges is malloc'd here; release it with wl_free.  route_ptr has n_trips+1 entries. */
int wl_route_trips(uint32_t n_nodes, const uint32_t *row_ptr, const uint32_t *head, const double *weight,
                   uint32_t n_trips, const uint32_t *origin, const uint32_t *dest, int n_threads,
                   uint64_t *route_ptr, uint32_t **out_route_edges)
{
    job J;
    memset(&J, 0, sizeof(J));
    J.n_nodes = n_nodes; J.row_ptr = row_ptr; J.head = head; J.w = weight;
    J.origin = origin; J.dest = dest;
    ki *s = (ki *)malloc(sizeof(ki) * (n_trips + 1));
    for (uint32_t i = 0; i < n_trips; i++) { s[i].key = origin[i]; s[i].idx = i; }
    qsort(s, n_trips, sizeof(ki), cmp_ki);
    uint32_t *sorted = (uint32_t *)malloc(sizeof(uint32_t) * (n_trips + 1));
    uint32_t *gp = (uint32_t *)malloc(sizeof(uint32_t) * (n_trips + 2));
    uint32_t ng = 0;
    for (uint32_t i = 0; i < n_trips; i++) {
        sorted[i] = s[i].idx;
        if (i == 0 || s[i].key != s[i - 1].key) gp[ng++] = i;
    }
    gp[ng] = n_trips;
    free(s);
    J.n_groups = ng; J.grp_ptr = gp; J.trip_sorted = sorted;
    J.route_len = (uint32_t *)calloc(n_trips + 1, sizeof(uint32_t));
    J.route_buf = (uint32_t **)calloc(n_trips + 1, sizeof(uint32_t *));
    pthread_mutex_init(&J.mu, NULL);
    if (n_threads < 1) n_threads = 1;
    if (n_threads > 256) n_threads = 256;
    pthread_t th[256];
    for (int k = 0; k < n_threads; k++) pthread_create(&th[k], NULL, worker, &J);
    for (int k = 0; k < n_threads; k++) pthread_join(th[k], NULL);
    uint64_t total = 0;
    for (uint32_t i = 0; i < n_trips; i++) { route_ptr[i] = total; total += J.route_len[i]; }
    route_ptr[n_trips] = total;
    uint32_t *all = (uint32_t *)malloc(sizeof(uint32_t) * (total + 1));
    for (uint32_t i = 0; i < n_trips; i++) {
        if (J.route_len[i]) memcpy(all + route_ptr[i], J.route_buf[i], sizeof(uint32_t) * J.route_len[i]);
        free(J.route_buf[i]);
    }
    *out_route_edges = all;
    free(J.route_len); free(J.route_buf); free(sorted); free(gp);
    pthread_mutex_destroy(&J.mu);
    return J.failed;
}

void wl_free(void *p) { free(p); }
