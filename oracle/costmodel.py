"""CPU oracle for the Advisor's cost model (PAPER.md:177-181 section 4.2, :303-321 section 5.3) -- TEST INFRASTRUCTURE ONLY.

Plain NumPy, float64, one statement per step of the paper's description; no blocking, no fusion.  Only tests/,
__graft_entry__.smoke() and bench.py's oracle legs may import this module; it imports nothing from the product.

What the paper fixes:
    MLP, "one input layer, four hidden layers, and one output layer"; hidden widths 2F, 4F, 2F, F for F input features
    (66, 132, 66, 33 for F = 33); Glorot initialisation [10]; bias 0; batch size 16; RMSprop, initial learning rate 0.01
    "stepped down by a factor of 0.1 every 30 epochs", weight decay 1e-4, 150 epochs; RMSE loss (Eq. 2); 80 % / 20 % split;
    Z-score standardisation; NRMSE = RMSE / (y_max - y_min) (Eq. 3), < 0.1 counts as success.
What it leaves open, and the reading taken (DESIGN.md Readings R20-R25):
    R20 activation: not stated -> ReLU after each of the four hidden layers, none on the output.
    R21 Glorot variant: uniform, W ~ U(-a, a), a = sqrt(6 / (fan_in + fan_out)); the uniforms u in [0, 1) are INPUTS.
    R22 RMSprop constants: smoothing 0.99, epsilon 1e-8 added outside the square root, no momentum, not centred; weight decay
        as an L2 term added to the gradient (g + wd * w), applied to weights and biases alike.
    R23 loss per mini-batch: RMSE over the samples of that batch; its gradient at RMSE == 0 is taken as 0.
    R24 batches: the order of the training samples in each epoch is an INPUT (one permutation per epoch); the last batch of an
        epoch may be short.
    R25 Z-score: features and target, with the mean and the population standard deviation (ddof = 0) of the TRAINING rows;
        a column with zero deviation is divided by 1.

Parameter packing (shared convention with the CUDA path, which implements it separately): for layer l = 0..4 with
n_in -> n_out, first the weight matrix W_l [n_out][n_in] row-major (y = W x + b), then the bias b_l [n_out]; layers in order.
"""
import numpy as np

RMSPROP_ALPHA = 0.99
RMSPROP_EPS = 1e-8


def layer_widths(f: int):
    """[F, 2F, 4F, 2F, F, 1] (multiples of the number of input features)."""
    return [f, 2 * f, 4 * f, 2 * f, f, 1]


def param_count(f: int) -> int:
    w = layer_widths(f)
    return sum(w[l + 1] * w[l] + w[l + 1] for l in range(5))


def glorot_init(f: int, uniforms: np.ndarray):
    """List of (W, b) from uniforms in [0, 1): one per weight, consumed in packing order; biases are 0."""
    w = layer_widths(f)
    u = np.asarray(uniforms, dtype=np.float64).reshape(-1)
    params, k = [], 0
    for l in range(5):
        n_in, n_out = w[l], w[l + 1]
        a = np.sqrt(6.0 / (n_in + n_out))
        W = (2.0 * u[k:k + n_in * n_out] - 1.0).reshape(n_out, n_in) * a
        k += n_in * n_out
        params.append((W, np.zeros(n_out)))
    return params


def pack(params) -> np.ndarray:
    return np.concatenate([np.concatenate([W.reshape(-1), b]) for W, b in params])


def unpack(f: int, flat):
    w = layer_widths(f)
    flat = np.asarray(flat, dtype=np.float64)
    params, k = [], 0
    for l in range(5):
        n_in, n_out = w[l], w[l + 1]
        W = flat[k:k + n_in * n_out].reshape(n_out, n_in).copy()
        k += n_in * n_out
        b = flat[k:k + n_out].copy()
        k += n_out
        params.append((W, b))
    return params


def forward(params, x):
    """x [n, F] -> (prediction [n], list of layer inputs a_0..a_4, list of pre-activations z_0..z_4)."""
    a = np.asarray(x, dtype=np.float64)
    acts, pre = [], []
    for l, (W, b) in enumerate(params):
        acts.append(a)
        z = a @ W.T + b
        pre.append(z)
        a = np.maximum(z, 0.0) if l < 4 else z
    return a[:, 0], acts, pre


def predict(params, x):
    return forward(params, x)[0]


def rmse(pred, y) -> float:
    """Eq. 2."""
    pred, y = np.asarray(pred, dtype=np.float64), np.asarray(y, dtype=np.float64)
    return float(np.sqrt(np.mean((pred - y) ** 2)))


def nrmse(pred, y) -> float:
    """Eq. 3: RMSE / (y_max - y_min)."""
    y = np.asarray(y, dtype=np.float64)
    return rmse(pred, y) / float(y.max() - y.min())


def loss_and_grads(params, x, y):
    """RMSE of the batch and its gradient with respect to every (W, b), by back-propagation."""
    pred, acts, pre = forward(params, x)
    n = len(y)
    loss = rmse(pred, y)
    if loss == 0.0:
        delta = np.zeros((n, 1))
    else:
        delta = ((pred - y) / (n * loss)).reshape(n, 1)  # d RMSE / d prediction
    grads = [None] * 5
    for l in range(4, -1, -1):
        W, _ = params[l]
        grads[l] = (delta.T @ acts[l], delta.sum(axis=0))
        if l > 0:
            delta = (delta @ W) * (pre[l - 1] > 0.0)
    return loss, grads


def rmsprop_step(params, state, grads, lr, weight_decay):
    """One RMSprop update in place (Reading R22): g += wd * p;  v = 0.99 v + 0.01 g^2;  p -= lr * g / (sqrt(v) + 1e-8)."""
    for l in range(5):
        for k in range(2):
            p, v, g = params[l][k], state[l][k], grads[l][k]
            g = g + weight_decay * p
            v *= RMSPROP_ALPHA
            v += (1.0 - RMSPROP_ALPHA) * g * g
            p -= lr * g / (np.sqrt(v) + RMSPROP_EPS)


def learning_rate(epoch: int, lr0=0.01, step=30, gamma=0.1) -> float:
    """0.01 stepped down by 0.1 every 30 epochs."""
    return lr0 * gamma ** (epoch // step)


def train(f, x, y, uniforms, perms, epochs=150, batch=16, lr0=0.01, step=30, gamma=0.1, weight_decay=1e-4, max_steps=None):
    """The training protocol of PAPER.md:305-307 on already standardised x [n, F], y [n].
    perms [epochs, n]: sample order of each epoch.  Returns (params, mean batch loss per epoch).  max_steps stops early
    (after that many updates in total), for step-by-step comparisons."""
    x, y = np.asarray(x, dtype=np.float64), np.asarray(y, dtype=np.float64)
    n = len(y)
    params = glorot_init(f, uniforms)
    state = [(np.zeros_like(W), np.zeros_like(b)) for W, b in params]
    epoch_loss, steps = [], 0
    for e in range(epochs):
        lr = learning_rate(e, lr0, step, gamma)
        order = np.asarray(perms[e], dtype=np.int64)
        losses = []
        for s in range(0, n, batch):
            if max_steps is not None and steps >= max_steps:
                break
            idx = order[s:s + batch]
            loss, grads = loss_and_grads(params, x[idx], y[idx])
            rmsprop_step(params, state, grads, lr, weight_decay)
            losses.append(loss)
            steps += 1
        epoch_loss.append(float(np.mean(losses)) if losses else float("nan"))
    return params, np.array(epoch_loss)


def zscore_fit(a):
    """Mean and population standard deviation per column (Reading R25); zero deviation -> 1."""
    a = np.asarray(a, dtype=np.float64)
    a2 = a.reshape(len(a), -1)
    mean = a2.mean(axis=0)
    std = np.sqrt(((a2 - mean) ** 2).mean(axis=0))
    std = np.where(std == 0.0, 1.0, std)
    return mean, std


def zscore_apply(a, mean, std):
    a = np.asarray(a, dtype=np.float64)
    return ((a.reshape(len(a), -1) - mean) / std).reshape(a.shape)
