"""Pins of the cost-model oracle (oracle/costmodel.py) against what the paper and the mathematics fix
(PAPER.md:305-321): architecture numbers the paper prints, Eq. 2 / Eq. 3 on a hand example, the learning-rate schedule,
finite differences for back-propagation, a closed form for the first RMSprop step, Glorot moments, and -- the strongest
one -- the whole training trajectory against torch's own Linear / RMSprop / StepLR on the CPU (a library routine the
oracle shares no code with).  CPU only."""
import numpy as np
import pytest

from oracle import costmodel as cm
from paper_2301_03636_b200 import inputs


def test_architecture_numbers_printed_in_the_paper():
    # "with 33 input features, have 66, 132, 66, and 33 neurons"
    assert cm.layer_widths(33) == [33, 66, 132, 66, 33, 1]
    # 33*66 + 66*132 + 132*66 + 66*33 + 33*1 weights, 66 + 132 + 66 + 33 + 1 biases
    assert cm.param_count(33) == 33 * 66 + 66 * 132 + 132 * 66 + 66 * 33 + 33 + (66 + 132 + 66 + 33 + 1)
    assert cm.param_count(5) == 20 * 25 + 10 * 5 + 1


def test_eq2_eq3_on_a_hand_example():
    pred, y = [1.0, 2.0, 3.0], [1.0, 2.0, 5.0]
    assert cm.rmse(pred, y) == pytest.approx(np.sqrt(4.0 / 3.0), rel=1e-15)          # Eq. 2
    assert cm.nrmse(pred, y) == pytest.approx(np.sqrt(4.0 / 3.0) / 4.0, rel=1e-15)   # Eq. 3: / (y_max - y_min)
    assert cm.rmse(y, y) == 0.0


def test_learning_rate_schedule():
    # "initial learning rate of 0.01 that is stepped down by a factor of 0.1 every 30 epochs ... for 150 epochs"
    want = {0: 1e-2, 29: 1e-2, 30: 1e-3, 59: 1e-3, 60: 1e-4, 90: 1e-5, 120: 1e-6, 149: 1e-6}
    for e, lr in want.items():
        assert cm.learning_rate(e) == pytest.approx(lr, rel=1e-12)


def test_glorot_bounds_moments_and_zero_bias():
    f = 12
    u = inputs.uniforms(7, cm.param_count(f))
    params = cm.glorot_init(f, u)
    w = cm.layer_widths(f)
    for l, (W, b) in enumerate(params):
        a = np.sqrt(6.0 / (w[l] + w[l + 1]))
        assert W.shape == (w[l + 1], w[l]) and not b.any()
        assert np.abs(W).max() <= a
        if W.size > 200:  # Var U(-a, a) = a^2 / 3 = 2 / (fan_in + fan_out)
            assert W.var() == pytest.approx(2.0 / (w[l] + w[l + 1]), rel=0.2)
            assert abs(W.mean()) < 3 * a / np.sqrt(3 * W.size)
    # u = 0 and u -> 1 map to the two ends of the interval, u = 0.5 to zero
    p0 = cm.glorot_init(f, np.zeros(cm.param_count(f)))
    assert p0[0][0][0, 0] == -np.sqrt(6.0 / (w[0] + w[1]))
    assert not cm.glorot_init(f, np.full(cm.param_count(f), 0.5))[2][0].any()


def test_pack_unpack_round_trip_and_order():
    f = 4
    params = cm.glorot_init(f, inputs.uniforms(3, cm.param_count(f)))
    params[0][1][:] = np.arange(2 * f) + 1.0
    flat = cm.pack(params)
    assert flat.size == cm.param_count(f)
    assert np.array_equal(flat[:2 * f * f], params[0][0].reshape(-1))           # W_0 row-major first
    assert np.array_equal(flat[2 * f * f:2 * f * f + 2 * f], params[0][1])      # then b_0
    back = cm.unpack(f, flat)
    for (W, b), (W2, b2) in zip(params, back):
        assert np.array_equal(W, W2) and np.array_equal(b, b2)


def test_backpropagation_against_central_finite_differences():
    f, n = 5, 7
    rng = np.random.default_rng(11)
    params = cm.glorot_init(f, inputs.uniforms(5, cm.param_count(f)))
    for _, b in params:
        b += 0.1 * rng.standard_normal(b.shape)  # non-zero biases so their gradient is exercised away from the start
    x, y = rng.standard_normal((n, f)), rng.standard_normal(n)
    loss, grads = cm.loss_and_grads(params, x, y)
    assert loss == pytest.approx(cm.rmse(cm.predict(params, x), y), rel=1e-15)
    flat = cm.pack(params)
    gflat = cm.pack(grads)
    h = 1e-6
    worst = 0.0
    for k in rng.choice(flat.size, size=120, replace=False):
        fp, fm = flat.copy(), flat.copy()
        fp[k] += h
        fm[k] -= h
        num = (cm.rmse(cm.predict(cm.unpack(f, fp), x), y) - cm.rmse(cm.predict(cm.unpack(f, fm), x), y)) / (2 * h)
        worst = max(worst, abs(num - gflat[k]))
    assert worst < 1e-8, worst
    # the loss is a function of the prediction only through the residual: zero residual -> zero gradient by Reading R23
    pred = cm.predict(params, x)
    _, g0 = cm.loss_and_grads(params, x, pred)
    assert not cm.pack(g0).any()


def test_first_rmsprop_step_closed_form():
    # v_1 = 0.01 g^2  =>  dp = -lr * g / (0.1 |g| + 1e-8): the first step has magnitude ~ 10 lr whatever the gradient's scale
    p = [(np.array([[2.0]]), np.array([-3.0]))] + [(np.zeros((1, 1)), np.zeros(1)) for _ in range(4)]
    st = [(np.zeros((1, 1)), np.zeros(1)) for _ in range(5)]
    g = [(np.array([[0.5]]), np.array([-4.0]))] + [(np.zeros((1, 1)), np.zeros(1)) for _ in range(4)]
    cm.rmsprop_step(p, st, g, lr=0.01, weight_decay=0.0)
    assert p[0][0][0, 0] == pytest.approx(2.0 - 0.01 * 0.5 / (0.1 * 0.5 + 1e-8), rel=1e-14)
    assert p[0][1][0] == pytest.approx(-3.0 + 0.01 * 4.0 / (0.1 * 4.0 + 1e-8), rel=1e-14)
    assert st[0][0][0, 0] == pytest.approx(0.01 * 0.25, rel=1e-14)
    # weight decay enters as g + wd * p (Reading R22): with g = 0 the step is -lr * sign(p) / (0.1 + 1e-8 / |wd p|)
    p = [(np.array([[2.0]]), np.array([0.0]))] + [(np.zeros((1, 1)), np.zeros(1)) for _ in range(4)]
    st = [(np.zeros((1, 1)), np.zeros(1)) for _ in range(5)]
    g = [(np.zeros((1, 1)), np.zeros(1)) for _ in range(5)]
    cm.rmsprop_step(p, st, g, lr=0.01, weight_decay=1e-4)
    assert p[0][0][0, 0] == pytest.approx(2.0 - 0.01 * 2e-4 / (0.1 * 2e-4 + 1e-8), rel=1e-14)


def test_zscore_statistics_and_degenerate_column():
    rng = np.random.default_rng(2)
    a = rng.standard_normal((50, 4)) * [1.0, 10.0, 0.1, 0.0] + [0.0, 5.0, -3.0, 7.0]
    mean, std = cm.zscore_fit(a)
    z = cm.zscore_apply(a, mean, std)
    assert np.allclose(z[:, :3].mean(axis=0), 0.0, atol=1e-13) and np.allclose(z[:, :3].std(axis=0), 1.0, atol=1e-13)
    assert std[3] == 1.0 and not z[:, 3].any()  # constant column: divided by 1
    assert std[1] == pytest.approx(a[:, 1].std(ddof=0), rel=1e-14)


def _torch_reference(f, x, y, uniforms, perms, epochs, batch, weight_decay):
    torch = pytest.importorskip("torch")
    torch.set_num_threads(1)
    w = cm.layer_widths(f)
    layers = []
    for l in range(5):
        layers.append(torch.nn.Linear(w[l], w[l + 1]).double())
        if l < 4:
            layers.append(torch.nn.ReLU())
    net = torch.nn.Sequential(*layers)
    lin = [m for m in net if isinstance(m, torch.nn.Linear)]
    u = torch.from_numpy(np.asarray(uniforms, dtype=np.float64))
    k = 0
    with torch.no_grad():
        for l, m in enumerate(lin):  # the same uniforms through torch's own xavier bound
            n = w[l] * w[l + 1]
            bound = torch.nn.init.calculate_gain("linear") * np.sqrt(6.0 / (w[l] + w[l + 1]))
            m.weight.copy_(((2.0 * u[k:k + n] - 1.0) * bound).reshape(w[l + 1], w[l]))
            m.bias.zero_()
            k += n
    opt = torch.optim.RMSprop(net.parameters(), lr=0.01, alpha=0.99, eps=1e-8, weight_decay=weight_decay)
    sched = torch.optim.lr_scheduler.StepLR(opt, step_size=30, gamma=0.1)
    xt, yt = torch.from_numpy(x), torch.from_numpy(y)
    losses = []
    for e in range(epochs):
        tot = []
        for s in range(0, len(y), batch):
            idx = torch.from_numpy(np.asarray(perms[e][s:s + batch], dtype=np.int64))
            opt.zero_grad()
            loss = torch.sqrt(torch.nn.functional.mse_loss(net(xt[idx])[:, 0], yt[idx]))
            loss.backward()
            opt.step()
            tot.append(float(loss.detach()))
        sched.step()
        losses.append(np.mean(tot))
    flat = np.concatenate([np.concatenate([m.weight.detach().numpy().reshape(-1), m.bias.detach().numpy()]) for m in lin])
    return flat, np.array(losses)


def test_training_trajectory_matches_torch_linear_rmsprop_steplr():
    """The oracle's hand-written forward / backward / RMSprop / schedule against torch's, same init, same batches, fp64,
    across two learning-rate steps (epochs 30 and 60) and with a short last batch (n = 37, batch 16)."""
    f, n, epochs = 3, 37, 65
    rng = np.random.default_rng(5)
    x = rng.standard_normal((n, f))
    y = np.tanh(x @ [1.0, -2.0, 0.5]) + 0.1 * rng.standard_normal(n)
    u = inputs.uniforms(9, cm.param_count(f))
    perms = inputs.permutations(9, epochs, n)
    params, losses = cm.train(f, x, y, u, perms, epochs=epochs)
    ref, ref_losses = _torch_reference(f, x, y, u, perms, epochs, 16, 1e-4)
    got = cm.pack(params)
    assert np.abs(got - ref).max() <= 1e-9 * max(1.0, np.abs(ref).max()), np.abs(got - ref).max()
    assert np.allclose(losses, ref_losses, rtol=1e-9, atol=1e-12)
    assert losses[-1] < 0.5 * losses[0]  # it learns


def test_training_reaches_the_papers_success_criterion_on_a_learnable_target():
    # a smooth function of the features: NRMSE < 0.1 on held-out rows, with the 80/20 split and Z-score
    f, n = 4, 400
    rng = np.random.default_rng(8)
    x = rng.uniform(-2, 2, size=(n, f))
    y = 3.0 * x[:, 0] - x[:, 1] * x[:, 2] + np.abs(x[:, 3])
    order = inputs.permutations(12, 1, n)[0]
    tr, va = order[:320], order[320:]
    mx, sx = cm.zscore_fit(x[tr])
    my, sy = cm.zscore_fit(y[tr])
    xs, ys = cm.zscore_apply(x, mx, sx), cm.zscore_apply(y, my, sy)
    params, losses = cm.train(f, xs[tr], ys[tr], inputs.uniforms(12, cm.param_count(f)), inputs.permutations(13, 60, 320), epochs=60)
    pred = cm.predict(params, xs[va]) * sy[0] + my[0]
    assert cm.nrmse(pred, y[va]) < 0.1
    assert losses[-1] < losses[0]


def test_max_steps_stops_after_that_many_updates():
    f, n = 3, 40
    rng = np.random.default_rng(1)
    x, y = rng.standard_normal((n, f)), rng.standard_normal(n)
    u, perms = inputs.uniforms(1, cm.param_count(f)), inputs.permutations(1, 3, n)
    p0 = cm.pack(cm.train(f, x, y, u, perms, epochs=3, max_steps=0)[0])
    assert np.array_equal(p0, cm.pack(cm.glorot_init(f, u)))
    p4 = cm.pack(cm.train(f, x, y, u, perms, epochs=3, max_steps=4)[0])  # 3 batches of epoch 0 + 1 of epoch 1
    q = cm.glorot_init(f, u)
    st = [(np.zeros_like(W), np.zeros_like(b)) for W, b in q]
    for idx in (perms[0][0:16], perms[0][16:32], perms[0][32:40], perms[1][0:16]):
        _, g = cm.loss_and_grads(q, x[idx], y[idx])
        cm.rmsprop_step(q, st, g, 0.01, 1e-4)
    assert np.array_equal(p4, cm.pack(q))
