/*
 * dqn_oracle.c -- CPU ORACLE of the DQN training step (test infrastructure only; see mig_oracle.h).
 *
 * the repartitioning policy is trained with "Deep Q-Learning, incorporating an epsilon-greedy
 * exploration-exploitation strategy and an experience replay buffer [21]"; L214: "discounted rewards over time".  The paper
 * gives no hyper-parameter, loss or optimiser; the readings taken are DESIGN.md #33-#36:
 *   network    Q(s) = b3 + relu(b2 + relu(b1 + s W1) W2) W3, W stored [in][out] (the C4 network)
 *   target     y_b = r_b + gamma (1 - done_b) max_a' Q_target(s'_b, a')           (frozen target network, Mnih et al. [21])
 *   loss       L = 1/(2B) sum_b (Q(s_b, a_b) - y_b)^2                             (plain squared TD error)
 *   optimiser  theta <- theta - lr dL/dtheta                                      (plain SGD)
 *   sampling   index_b = (w * size) >> 32, w = word 0 of Philox4x32-10(counter (b, 3, step, 0), key = seed): stream 3
 * Everything is double precision, plain loops, in the order of the formulas above.  Shares no code with the CUDA path.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include "mig_oracle.h"

struct orc_dqn {
  uint32_t H, A;
  double gamma, lr;
  double *w[2];   /* [0] online, [1] target: flat W1 [64][H], b1 [H], W2 [H][H], b2 [H], W3 [H][A], b3 [A] */
  size_t n;       /* parameters per network */
};

static size_t off_b1(uint32_t H) { return (size_t)ORC_STATE_DIM * H; }
static size_t off_W2(uint32_t H) { return off_b1(H) + H; }
static size_t off_b2(uint32_t H) { return off_W2(H) + (size_t)H * H; }
static size_t off_W3(uint32_t H) { return off_b2(H) + H; }
static size_t off_b3(uint32_t H, uint32_t A) { return off_W3(H) + (size_t)H * A; }

size_t orc_dqn_n_params(uint32_t H, uint32_t A) { return off_b3(H, A) + A; }

orc_dqn_t *orc_dqn_create(const orc_qnet_t *init, double gamma, double lr)
{
  orc_dqn_t *d = (orc_dqn_t *)calloc(1, sizeof(*d));
  d->H = init->hidden; d->A = init->n_actions; d->gamma = gamma; d->lr = lr;
  d->n = orc_dqn_n_params(d->H, d->A);
  const float *src[6] = { init->W1, init->b1, init->W2, init->b2, init->W3, init->b3 };
  size_t sz[6] = { (size_t)ORC_STATE_DIM * d->H, d->H, (size_t)d->H * d->H, d->H, (size_t)d->H * d->A, d->A };
  for (int k = 0; k < 2; ++k) {
    d->w[k] = (double *)malloc(sizeof(double) * d->n);
    size_t o = 0;
    for (int i = 0; i < 6; ++i) { for (size_t j = 0; j < sz[i]; ++j) d->w[k][o + j] = (double)src[i][j]; o += sz[i]; }
  }
  return d;
}

void orc_dqn_destroy(orc_dqn_t *d) { if (!d) return; free(d->w[0]); free(d->w[1]); free(d); }
void orc_dqn_sync_target(orc_dqn_t *d) { memcpy(d->w[1], d->w[0], sizeof(double) * d->n); }
void orc_dqn_get(const orc_dqn_t *d, int which, double *flat) { memcpy(flat, d->w[which ? 1 : 0], sizeof(double) * d->n); }
void orc_dqn_set(orc_dqn_t *d, int which, const double *flat) { memcpy(d->w[which ? 1 : 0], flat, sizeof(double) * d->n); }

/* forward of one state through the network `w`; keeps the hidden activations */
static void forward(const orc_dqn_t *d, const double *w, const float *s, double *h1, double *h2, double *q)
{
  uint32_t H = d->H, A = d->A;
  const double *W1 = w, *b1 = w + off_b1(H), *W2 = w + off_W2(H), *b2 = w + off_b2(H), *W3 = w + off_W3(H), *b3 = w + off_b3(H, A);
  for (uint32_t n = 0; n < H; ++n) { double z = b1[n]; for (uint32_t k = 0; k < ORC_STATE_DIM; ++k) z += (double)s[k] * W1[(size_t)k * H + n]; h1[n] = z > 0 ? z : 0; }
  for (uint32_t n = 0; n < H; ++n) { double z = b2[n]; for (uint32_t k = 0; k < H; ++k) z += h1[k] * W2[(size_t)k * H + n]; h2[n] = z > 0 ? z : 0; }
  for (uint32_t n = 0; n < A; ++n) { double z = b3[n]; for (uint32_t k = 0; k < H; ++k) z += h2[k] * W3[(size_t)k * A + n]; q[n] = z; }
}

/* Q-values of the online (which = 0) or target (1) network, double */
void orc_dqn_q(const orc_dqn_t *d, int which, const float *s, uint32_t B, double *q_out)
{
  double *h1 = (double *)malloc(sizeof(double) * d->H), *h2 = (double *)malloc(sizeof(double) * d->H);
  for (uint32_t b = 0; b < B; ++b) forward(d, d->w[which ? 1 : 0], s + (size_t)b * ORC_STATE_DIM, h1, h2, q_out + (size_t)b * d->A);
  free(h1); free(h2);
}

/* loss and its gradient with respect to the ONLINE parameters (grad: n_params doubles, same flat order; may be NULL) */
double orc_dqn_loss_grad(const orc_dqn_t *d, const float *s, const uint8_t *a, const float *r, const float *s2,
                         const uint8_t *done, uint32_t B, double *grad)
{
  uint32_t H = d->H, A = d->A;
  const double *w = d->w[0];
  const double *W2 = w + off_W2(H), *W3 = w + off_W3(H);
  double *h1 = (double *)malloc(sizeof(double) * H), *h2 = (double *)malloc(sizeof(double) * H), *q = (double *)malloc(sizeof(double) * A);
  double *t1 = (double *)malloc(sizeof(double) * H), *t2 = (double *)malloc(sizeof(double) * H), *qt = (double *)malloc(sizeof(double) * A);
  double *dz2 = (double *)malloc(sizeof(double) * H), *dz1 = (double *)malloc(sizeof(double) * H);
  if (grad) memset(grad, 0, sizeof(double) * d->n);
  double loss = 0.0;
  for (uint32_t b = 0; b < B; ++b) {
    const float *x = s + (size_t)b * ORC_STATE_DIM;
    forward(d, w, x, h1, h2, q);
    forward(d, d->w[1], s2 + (size_t)b * ORC_STATE_DIM, t1, t2, qt);
    double mx = qt[0]; for (uint32_t n = 1; n < A; ++n) if (qt[n] > mx) mx = qt[n];
    double y = (double)r[b] + ((done && done[b]) ? 0.0 : d->gamma * mx);       /* TD target, target network frozen */
    double delta = q[a[b]] - y;
    loss += delta * delta / (2.0 * (double)B);
    if (!grad) continue;
    double g = delta / (double)B;                                               /* dL/dQ(s_b, a_b) */
    double *gW1 = grad, *gb1 = grad + off_b1(H), *gW2 = grad + off_W2(H), *gb2 = grad + off_b2(H), *gW3 = grad + off_W3(H), *gb3 = grad + off_b3(H, A);
    gb3[a[b]] += g;
    for (uint32_t k = 0; k < H; ++k) gW3[(size_t)k * A + a[b]] += h2[k] * g;
    for (uint32_t k = 0; k < H; ++k) dz2[k] = h2[k] > 0 ? g * W3[(size_t)k * A + a[b]] : 0.0;      /* relu' */
    for (uint32_t k = 0; k < H; ++k) { gb2[k] += dz2[k]; }
    for (uint32_t i = 0; i < H; ++i) for (uint32_t k = 0; k < H; ++k) gW2[(size_t)i * H + k] += h1[i] * dz2[k];
    for (uint32_t i = 0; i < H; ++i) { double acc = 0.0; for (uint32_t k = 0; k < H; ++k) acc += dz2[k] * W2[(size_t)i * H + k]; dz1[i] = h1[i] > 0 ? acc : 0.0; }
    for (uint32_t i = 0; i < H; ++i) gb1[i] += dz1[i];
    for (uint32_t j = 0; j < ORC_STATE_DIM; ++j) for (uint32_t i = 0; i < H; ++i) gW1[(size_t)j * H + i] += (double)x[j] * dz1[i];
  }
  free(h1); free(h2); free(q); free(t1); free(t2); free(qt); free(dz2); free(dz1);
  return loss;
}

/* one SGD step on the batch; returns the loss BEFORE the step */
double orc_dqn_train_step(orc_dqn_t *d, const float *s, const uint8_t *a, const float *r, const float *s2, const uint8_t *done, uint32_t B)
{
  double *g = (double *)malloc(sizeof(double) * d->n);
  double loss = orc_dqn_loss_grad(d, s, a, r, s2, done, B, g);
  for (size_t i = 0; i < d->n; ++i) d->w[0][i] -= d->lr * g[i];
  free(g);
  return loss;
}

/* uniform sampling with replacement from the first `size` transitions of the replay buffer (reading #36) */
void orc_replay_sample(uint64_t seed, uint32_t step, uint32_t size, uint32_t B, uint32_t *idx_out)
{
  for (uint32_t b = 0; b < B; ++b) {
    uint32_t w[4];
    orc_philox4x32_10(b, 3u, step, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), w);
    idx_out[b] = (uint32_t)(((uint64_t)w[0] * size) >> 32);
  }
}
