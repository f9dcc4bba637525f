/* vmat_oracle_mt.c - the all-cores variant of the CPU oracle for the TIMED CPU BASELINE (bench.py `cpu_baseline`
 * second leg, SURVEY.md 8(d) "CPU baseline" (ii)) - TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * PAPER.md L191 (strategy S3): the paper's own CPU run splits the work over pthreads (4 cores / 8 threads).  This file
 * does the same with the plain oracle: it adds NO arithmetic of its own - every thread calls the single-thread
 * functions of vmat_oracle.c (oracle_dose, oracle_objective_grad, oracle_price, oracle_select_rows) on its share:
 *   O1 / O3  the COO range is cut into n_threads consecutive pieces, each thread sums its piece into a private
 *            FP64 vector, the private vectors are added in thread order (piece-additivity of a sum over triplets;
 *            the angle-block case is pin P6, L119);
 *   O2       the voxel range is cut into pieces, F = the pieces' partial sums added in thread order;
 *   O4       the leaf rows are cut into pieces (rows are independent, L133): bit-identical to the single thread.
 * O5 is not threaded.  Pin (tests/test_oracle_mt.py): every output equals the single-thread oracle's to 1e-12
 * relative (the sums differ by the order of FP64 additions only), leaf positions and row prices bit for bit.
 * It is linked together with vmat_oracle.c into libvmat_oracle_mt.so; the plain oracle library does not contain it. */
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

void oracle_dose(int64_t nnz, const int32_t *coo_voxel, const int32_t *coo_beamlet, const float *coo_val,
                 int32_t n_voxels, const float *x, double *d);
double oracle_objective_grad(int32_t n_voxels, const double *d, const uint8_t *voxel_struct, const float *T,
                             const float *w_over, const float *w_under, double *g);
void oracle_price(int64_t nnz, const int32_t *coo_voxel, const int32_t *coo_beamlet, const float *coo_val,
                  int32_t n_beamlets, const double *g, double *p);
void oracle_select_rows(int32_t n_rows, const int32_t *leafrow_col_offset, const float *p, int32_t *Lout,
                        int32_t *Rout, double *row_price, double *S);

typedef struct {
    int kind;                   /* 0 dose, 1 price, 2 objective, 3 select, 4 add the private vectors over a range */
    int t, n_threads;
    int64_t nnz;
    const int32_t *vox, *beam;
    const float *val;
    int32_t n_out;              /* length of the output vector of kinds 0, 1, 4 */
    const float *x;             /* dose */
    const double *g_in;         /* price */
    double *priv;               /* [n_threads][n_out] private vectors */
    double *out;
    /* objective */
    const double *d;
    const uint8_t *sid;
    const float *T, *wo, *wu;
    double *g_out, F_part;
    /* selection */
    int32_t n_rows;
    const int32_t *lco;
    const float *p32;
    int32_t *L, *R;
    double *rp;
    int32_t max_n;
} job_t;

static void range_of(int64_t n, int t, int nt, int64_t *a, int64_t *b)
{
    *a = n * t / nt;
    *b = n * (t + 1) / nt;
}

static void *worker(void *arg)
{
    job_t *j = (job_t *)arg;
    int64_t a, b;
    switch (j->kind) {
    case 0:
        range_of(j->nnz, j->t, j->n_threads, &a, &b);
        oracle_dose(b - a, j->vox + a, j->beam + a, j->val + a, j->n_out, j->x, j->priv + (size_t)j->t * j->n_out);
        break;
    case 1:
        range_of(j->nnz, j->t, j->n_threads, &a, &b);
        oracle_price(b - a, j->vox + a, j->beam + a, j->val + a, j->n_out, j->g_in, j->priv + (size_t)j->t * j->n_out);
        break;
    case 2:
        range_of(j->n_out, j->t, j->n_threads, &a, &b);
        j->F_part = oracle_objective_grad((int32_t)(b - a), j->d + a, j->sid + a, j->T, j->wo, j->wu, j->g_out + a);
        break;
    case 3: {
        range_of(j->n_rows, j->t, j->n_threads, &a, &b);
        double *S = (double *)malloc(((size_t)j->max_n + 1) * sizeof(double));
        oracle_select_rows((int32_t)(b - a), j->lco + a, j->p32, j->L + a, j->R + a, j->rp + a, S);
        free(S);
        break;
    }
    case 4:
        range_of(j->n_out, j->t, j->n_threads, &a, &b);
        for (int64_t i = a; i < b; ++i) {
            double s = 0.0;
            for (int q = 0; q < j->n_threads; ++q) s += j->priv[(size_t)q * j->n_out + i];   /* thread order */
            j->out[i] = s;
        }
        break;
    }
    return NULL;
}

static void run(job_t *proto, int n_threads)
{
    pthread_t *th = (pthread_t *)malloc(sizeof(pthread_t) * (size_t)n_threads);
    job_t *jobs = (job_t *)malloc(sizeof(job_t) * (size_t)n_threads);
    for (int t = 0; t < n_threads; ++t) {
        jobs[t] = *proto;
        jobs[t].t = t;
        jobs[t].n_threads = n_threads;
        pthread_create(&th[t], NULL, worker, &jobs[t]);
    }
    for (int t = 0; t < n_threads; ++t) pthread_join(th[t], NULL);
    if (proto->kind == 2) {
        double F = 0.0;
        for (int t = 0; t < n_threads; ++t) F += jobs[t].F_part;                                /* thread order */
        proto->F_part = F;
    }
    free(jobs);
    free(th);
}

/* priv: caller scratch of n_threads * n_voxels doubles */
void oracle_mt_dose(int n_threads, int64_t nnz, const int32_t *vox, const int32_t *beam, const float *val,
                    int32_t n_voxels, const float *x, double *d, double *priv)
{
    job_t j;
    memset(&j, 0, sizeof(j));
    j.kind = 0; j.nnz = nnz; j.vox = vox; j.beam = beam; j.val = val; j.n_out = n_voxels; j.x = x; j.priv = priv;
    run(&j, n_threads);
    j.kind = 4; j.out = d;
    run(&j, n_threads);
}

/* priv: caller scratch of n_threads * n_beamlets doubles */
void oracle_mt_price(int n_threads, int64_t nnz, const int32_t *vox, const int32_t *beam, const float *val,
                     int32_t n_beamlets, const double *g, double *p, double *priv)
{
    job_t j;
    memset(&j, 0, sizeof(j));
    j.kind = 1; j.nnz = nnz; j.vox = vox; j.beam = beam; j.val = val; j.n_out = n_beamlets; j.g_in = g; j.priv = priv;
    run(&j, n_threads);
    j.kind = 4; j.out = p;
    run(&j, n_threads);
}

double oracle_mt_objective_grad(int n_threads, int32_t n_voxels, const double *d, const uint8_t *sid, const float *T,
                                const float *wo, const float *wu, double *g)
{
    job_t j;
    memset(&j, 0, sizeof(j));
    j.kind = 2; j.n_out = n_voxels; j.d = d; j.sid = sid; j.T = T; j.wo = wo; j.wu = wu; j.g_out = g;
    run(&j, n_threads);
    return j.F_part;
}

void oracle_mt_select_rows(int n_threads, int32_t n_rows, const int32_t *lco, const float *p, int32_t *L, int32_t *R,
                           double *rp, int32_t max_n)
{
    job_t j;
    memset(&j, 0, sizeof(j));
    j.kind = 3; j.n_rows = n_rows; j.lco = lco; j.p32 = p; j.L = L; j.R = R; j.rp = rp; j.max_n = max_n;
    run(&j, n_threads);
}
