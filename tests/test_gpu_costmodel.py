"""GPU parity of the cost-model kernels (include/advisor_costmodel.h, through the ctypes binding) against oracle/costmodel.py
on the same seeded inputs.  Tolerances: the two sides differ only in floating-point summation order
(fp64).  Initialisation is bit-exact; after k <= 5 updates parameters agree to 1e-12; over whole trajectories (hundreds of
updates, each feeding the next through RMSprop's normalised step) to 1e-8 -- the oracle itself agrees with torch's
Linear/RMSprop/StepLR to 1e-9 over such a trajectory (tests/test_oracle_costmodel_pins.py)."""
import numpy as np
import pytest

from paper_2301_03636_b200 import inputs

pytestmark = pytest.mark.gpu

TOL_FEW_STEPS = 1e-12
TOL_TRAJECTORY = 1e-8


@pytest.fixture(scope="module")
def env():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from oracle import costmodel as cm
    from paper_2301_03636_b200 import binding as B
    from paper_2301_03636_b200 import costmodel as C

    class E:
        pass
    e = E()
    e.torch, e.cm, e.B, e.C = torch, cm, B, C
    e.dev = torch.device("cuda:0")
    return e


def _data(f, n, seed):
    rng = np.random.default_rng(seed)
    x = rng.standard_normal((n, f))
    y = np.tanh(x @ rng.standard_normal(f)) + 0.1 * rng.standard_normal(n)
    return x, y


def _gpu_train(env, f, x, y, u, perms, cluster, n_models=1, **kw):
    t = env.torch
    model = env.C.CostModel(f)
    xs, ys = t.from_numpy(x).to(env.dev), t.from_numpy(y).to(env.dev)
    ud = t.from_numpy(np.ascontiguousarray(u, dtype=np.float64).reshape(n_models, -1)).to(env.dev)
    pd = t.from_numpy(np.ascontiguousarray(perms, dtype=np.int32)).to(env.dev)
    params, loss = model.train(xs, ys, ud, pd, cluster_size=cluster, **kw)
    t.cuda.synchronize()
    return params.cpu().numpy(), loss.cpu().numpy()


def _rel(got, ref):
    return float(np.abs(got - ref).max() / max(1.0, np.abs(ref).max()))


@pytest.mark.parametrize("cluster", [1, 2, 4, 8])
@pytest.mark.parametrize("f,n,batch", [(3, 37, 16), (5, 40, 16), (12, 50, 7), (1, 9, 4)])
def test_initialisation_is_bit_exact_and_first_steps_match(env, f, n, batch, cluster):
    cm = env.cm
    x, y = _data(f, n, 100 + f)
    nw = env.C.costmodel_weight_count(f)
    assert nw == sum(a * b for a, b in zip(cm.layer_widths(f)[:-1], cm.layer_widths(f)[1:]))
    assert env.C.costmodel_param_count(f) == cm.param_count(f)
    u = inputs.uniforms(f, nw)
    epochs = 3
    perms = inputs.permutations(f, epochs, n)
    for k in (0, 1, 2, 5):
        got, _ = _gpu_train(env, f, x, y, u, perms, cluster, epochs=epochs, batch=batch, max_steps=k)
        ref = cm.pack(cm.train(f, x, y, u, perms, epochs=epochs, batch=batch, max_steps=k)[0])
        if k == 0:
            assert np.array_equal(got[0], ref)  # Glorot: (2u - 1) * sqrt(6 / (fan_in + fan_out)), biases 0
        else:
            assert _rel(got[0], ref) <= TOL_FEW_STEPS, (k, _rel(got[0], ref))


@pytest.mark.parametrize("cluster", [1, 2, 4, 8])
def test_whole_trajectory_matches_the_oracle_across_two_learning_rate_steps(env, cluster):
    # the configuration of the oracle's torch pin: n = 37 (short last batch), 65 epochs = 195 updates, lr steps at 30 and 60
    cm = env.cm
    f, n, epochs = 3, 37, 65
    rng = np.random.default_rng(5)
    x = rng.standard_normal((n, f))
    y = np.tanh(x @ [1.0, -2.0, 0.5]) + 0.1 * rng.standard_normal(n)
    u = inputs.uniforms(9, cm.param_count(f))[:env.C.costmodel_weight_count(f)]
    perms = inputs.permutations(9, epochs, n)
    got, loss = _gpu_train(env, f, x, y, u, perms, cluster, epochs=epochs)
    ref, ref_loss = cm.train(f, x, y, u, perms, epochs=epochs)
    assert _rel(got[0], cm.pack(ref)) <= TOL_TRAJECTORY, _rel(got[0], cm.pack(ref))
    assert np.allclose(loss[0], ref_loss, rtol=TOL_TRAJECTORY, atol=1e-12)
    assert loss[0, -1] < 0.5 * loss[0, 0]


@pytest.mark.parametrize("cluster", [0, 4, 8])
def test_the_papers_33_feature_network(env, cluster):
    # F = 33: 66, 132, 66, 33 hidden neurons; 22 111 parameters; needs >= 4 blocks' shared memory
    cm = env.cm
    f, n, epochs = 33, 100, 3
    x, y = _data(f, n, 33)
    u = inputs.uniforms(33, env.C.costmodel_weight_count(f))
    perms = inputs.permutations(33, epochs, n)
    got, loss = _gpu_train(env, f, x, y, u, perms, cluster, epochs=epochs)
    ref, ref_loss = cm.train(f, x, y, u, perms, epochs=epochs)
    assert got.shape == (1, 22111)
    assert _rel(got[0], cm.pack(ref)) <= TOL_TRAJECTORY, _rel(got[0], cm.pack(ref))
    assert np.allclose(loss[0], ref_loss, rtol=TOL_TRAJECTORY)


def test_shared_memory_limits_are_reported_not_worked_around(env):
    C, B = env.C, env.B
    assert C.costmodel_train_smem_bytes(33, 16, 1) > 232448 and C.costmodel_train_smem_bytes(33, 16, 2) > 232448
    assert 0 < C.costmodel_train_smem_bytes(33, 16, 4) <= 232448
    assert C.costmodel_train_smem_bytes(33, 16, 3) == 0 and C.costmodel_train_smem_bytes(0, 16, 1) == 0
    t = env.torch
    f, n = 33, 20
    x, y = _data(f, n, 1)
    xs, ys = t.from_numpy(x).to(env.dev), t.from_numpy(y).to(env.dev)
    u = t.from_numpy(inputs.uniforms(1, C.costmodel_weight_count(f))).to(env.dev)
    p = t.from_numpy(inputs.permutations(1, 1, n)).to(env.dev)
    out = t.empty(C.costmodel_param_count(f), dtype=t.float64, device=env.dev)
    args = [f, n, xs.data_ptr(), ys.data_ptr(), u.data_ptr(), p.data_ptr(), 1, 16, 0.01, 30, 0.1, 1e-4, -1, 1, 1, out.data_ptr(), 0, 0]
    assert C.costmodel_train_status(*args) == B.DSLASH_ERR_UNSUPPORTED          # one block cannot hold F = 33
    args[14] = 3
    assert C.costmodel_train_status(*args) == B.DSLASH_ERR_UNSUPPORTED          # cluster size not in {0,1,2,4,8}
    args[14] = 0
    for pos, bad, want in [(2, 0, B.DSLASH_ERR_NULL), (15, 0, B.DSLASH_ERR_NULL), (5, 0, B.DSLASH_ERR_NULL),
                           (0, 0, B.DSLASH_ERR_DIMS), (1, 0, B.DSLASH_ERR_DIMS), (7, 65, B.DSLASH_ERR_DIMS), (7, 0, B.DSLASH_ERR_DIMS),
                           (13, 0, B.DSLASH_ERR_DIMS), (6, -1, B.DSLASH_ERR_DIMS), (2, xs.data_ptr() + 4, B.DSLASH_ERR_ALIGN)]:
        a = list(args)
        a[pos] = bad
        assert C.costmodel_train_status(*a) == want, (pos, bad)
    a = list(args)
    a[6], a[9] = 100, 1  # 100 learning-rate steps > 32
    assert C.costmodel_train_status(*a) == B.DSLASH_ERR_UNSUPPORTED


def test_independent_models_in_one_launch_and_run_to_run_determinism(env):
    cm = env.cm
    f, n, epochs, m = 6, 45, 4, 5
    x, y = _data(f, n, 6)
    nw = env.C.costmodel_weight_count(f)
    u = np.stack([inputs.uniforms(60 + k, nw) for k in range(m)])
    perms = np.stack([inputs.permutations(60 + k, epochs, n) for k in range(m)])
    got, loss = _gpu_train(env, f, x, y, u, perms, 2, n_models=m, epochs=epochs)
    again, _ = _gpu_train(env, f, x, y, u, perms, 2, n_models=m, epochs=epochs)
    assert np.array_equal(got, again)
    for k in range(m):
        one, one_loss = _gpu_train(env, f, x, y, u[k], perms[k], 2, epochs=epochs)
        assert np.array_equal(one[0], got[k]) and np.array_equal(one_loss[0], loss[k])
        ref, ref_loss = cm.train(f, x, y, u[k], perms[k], epochs=epochs)
        assert _rel(got[k], cm.pack(ref)) <= TOL_TRAJECTORY
        assert np.allclose(loss[k], ref_loss, rtol=TOL_TRAJECTORY)
    assert not np.array_equal(got[0], got[1])


def test_epochs_without_updates_report_nan_and_zero_epochs_returns_the_initialisation(env):
    cm = env.cm
    f, n = 4, 20
    x, y = _data(f, n, 4)
    u = inputs.uniforms(4, env.C.costmodel_weight_count(f))
    perms = inputs.permutations(4, 3, n)
    got, loss = _gpu_train(env, f, x, y, u, perms, 1, epochs=3, max_steps=3)  # 2 batches in epoch 0, 1 in epoch 1, none in epoch 2
    ref, ref_loss = cm.train(f, x, y, u, perms, epochs=3, max_steps=3)
    assert _rel(got[0], cm.pack(ref)) <= TOL_FEW_STEPS
    assert np.isnan(loss[0, 2]) and np.isnan(ref_loss[2])
    assert np.allclose(loss[0, :2], ref_loss[:2], rtol=1e-12)
    got0, _ = _gpu_train(env, f, x, y, u, perms, 1, epochs=0)
    assert np.array_equal(got0[0], cm.pack(cm.glorot_init(f, u)))


def test_zero_residual_gives_zero_gradient(env):
    # Reading R23: RMSE == 0 -> gradient 0; with weight decay 0 the parameters must not move (and must not become NaN)
    cm = env.cm
    f, n = 2, 16
    x = np.zeros((n, f))
    y = np.zeros(n)  # zero inputs, zero biases -> prediction exactly 0 = y
    u = inputs.uniforms(2, env.C.costmodel_weight_count(f))
    perms = inputs.permutations(2, 2, n)
    got, loss = _gpu_train(env, f, x, y, u, perms, 1, epochs=2, weight_decay=0.0)
    assert np.array_equal(got[0], cm.pack(cm.glorot_init(f, u)))
    assert not loss.any()


@pytest.mark.parametrize("f,n,m", [(3, 1, 1), (5, 16, 2), (12, 1000, 1), (33, 531, 3)])
def test_predict_matches_the_oracle(env, f, n, m):
    cm, t = env.cm, env.torch
    rng = np.random.default_rng(f)
    x = rng.standard_normal((n, f))
    flats = []
    for k in range(m):
        params = cm.glorot_init(f, inputs.uniforms(k, cm.param_count(f)))
        for _, b in params:
            b += 0.3 * rng.standard_normal(b.shape)
        flats.append(cm.pack(params))
    model = env.C.CostModel(f)
    pred = model.predict(t.from_numpy(x).to(env.dev), t.from_numpy(np.stack(flats)).to(env.dev)).cpu().numpy()
    for k in range(m):
        ref = cm.predict(cm.unpack(f, flats[k]), x)
        assert np.abs(pred[k] - ref).max() <= 1e-13 * max(1.0, np.abs(ref).max())


def test_zscore_and_errors_match_the_oracle(env):
    cm, t = env.cm, env.torch
    rng = np.random.default_rng(2)
    n, f = 1237, 5
    a = rng.standard_normal((n, f)) * [1.0, 10.0, 0.1, 0.0, 1e3] + [0.0, 5.0, -3.0, 7.0, 1e6]
    yv = rng.standard_normal(n) * 4.0 + 2.0
    model = env.C.CostModel(f)
    ad, yd = t.from_numpy(a).to(env.dev), t.from_numpy(yv).to(env.dev)
    model.fit_scaler(ad, yd)
    mean, std = cm.zscore_fit(a)
    assert np.allclose(model.x_mean.cpu().numpy(), mean, rtol=1e-14, atol=1e-14)
    assert np.allclose(model.x_std.cpu().numpy(), std, rtol=1e-12)
    assert model.x_std.cpu().numpy()[3] == 1.0  # constant column: divided by 1 (Reading R25)
    z = model.scale_x(ad).cpu().numpy()
    assert np.allclose(z, cm.zscore_apply(a, mean, std), rtol=1e-9, atol=1e-9)
    assert not z[:, 3].any()
    my, sy = cm.zscore_fit(yv)
    zy = model.scale_y(yd)
    assert np.allclose(zy.cpu().numpy(), cm.zscore_apply(yv, my, sy), rtol=1e-12, atol=1e-13)
    back = model.scale_y(zy, inverse=True).cpu().numpy()
    assert np.allclose(back, yv, rtol=1e-13, atol=1e-13)
    pred = yv + rng.standard_normal(n)
    out = model.error(t.from_numpy(pred).to(env.dev), yd).cpu().numpy()
    assert out[0] == pytest.approx(cm.rmse(pred, yv), rel=1e-13)
    assert out[1] == pytest.approx(cm.nrmse(pred, yv), rel=1e-13)
    # Eq. 2 / Eq. 3 on the hand example of the oracle's pin
    out = model.error(t.tensor([1.0, 2.0, 3.0], dtype=t.float64, device=env.dev),
                      t.tensor([1.0, 2.0, 5.0], dtype=t.float64, device=env.dev)).cpu().numpy()
    assert out[0] == pytest.approx(np.sqrt(4.0 / 3.0), rel=1e-15) and out[1] == pytest.approx(np.sqrt(4.0 / 3.0) / 4.0, rel=1e-15)


def test_protocol_end_to_end_reaches_the_papers_success_criterion(env):
    """80/20 split, Z-score on the training rows, the paper's optimiser settings, NRMSE < 0.1 on the held-out rows
     -- all on the device -- and the same numbers as the oracle running the same protocol."""
    cm, t = env.cm, env.torch
    f, n, epochs = 4, 400, 60
    rng = np.random.default_rng(8)
    x = rng.uniform(-2, 2, size=(n, f))
    y = 3.0 * x[:, 0] - x[:, 1] * x[:, 2] + np.abs(x[:, 3])
    order = inputs.permutations(12, 1, n)[0]
    tr, va = order[:320], order[320:]
    u = inputs.uniforms(12, cm.param_count(f))[:env.C.costmodel_weight_count(f)]
    perms = inputs.permutations(13, epochs, 320)
    # device
    model = env.C.CostModel(f)
    xd, yd = t.from_numpy(x).to(env.dev), t.from_numpy(y).to(env.dev)
    xtr, ytr, xva, yva = xd[tr].contiguous(), yd[tr].contiguous(), xd[va].contiguous(), yd[va].contiguous()
    model.fit_scaler(xtr, ytr)
    params, loss = model.train(model.scale_x(xtr), model.scale_y(ytr), t.from_numpy(u).to(env.dev)[None], t.from_numpy(perms).to(env.dev),
                               epochs=epochs)
    pred = model.scale_y(model.predict(model.scale_x(xva))[0].contiguous(), inverse=True)
    rmse_gpu, nrmse_gpu = model.error(pred, yva).cpu().numpy()
    # oracle
    mx, sx = cm.zscore_fit(x[tr])
    my, sy = cm.zscore_fit(y[tr])
    xs, ys = cm.zscore_apply(x, mx, sx), cm.zscore_apply(y, my, sy)
    ref, ref_loss = cm.train(f, xs[tr], ys[tr], u, perms, epochs=epochs)
    ref_pred = cm.predict(ref, xs[va]) * sy[0] + my[0]
    assert nrmse_gpu < 0.1
    assert nrmse_gpu == pytest.approx(cm.nrmse(ref_pred, y[va]), rel=1e-6)
    assert np.allclose(loss.cpu().numpy()[0], ref_loss, rtol=1e-6)
    assert _rel(params.cpu().numpy()[0], cm.pack(ref)) <= 1e-6  # 1200 updates: looser than TOL_TRAJECTORY (195 updates)
