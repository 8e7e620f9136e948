"""Thin ctypes binding of the costmodel_* calls of libdslash_b200.so: the same names as include/advisor_costmodel.h,
argument marshalling only.  Every step (Glorot initialisation, forward, back-propagation, RMSprop, learning-rate schedule,
Z-score, RMSE / NRMSE) runs in the library's CUDA kernels; there is no Python or CPU fallback.

Pointers are plain integers (`tensor.data_ptr()`), streams the integer value of a cudaStream_t.  `CostModel` at the bottom
is the torch plumbing (device buffers, copies) for a caller that holds NumPy arrays.
"""
import ctypes

from . import binding as _B

_vp = ctypes.c_void_p
_i, _d, _ll = ctypes.c_int, ctypes.c_double, ctypes.c_longlong

# name -> (restype, argtypes); mirrors include/advisor_costmodel.h one to one
SIGNATURES = {
    "costmodel_param_count": (ctypes.c_size_t, [_i]),
    "costmodel_weight_count": (ctypes.c_size_t, [_i]),
    "costmodel_train_smem_bytes": (ctypes.c_size_t, [_i, _i, _i]),
    "costmodel_train": (_i, [_i, _i, _vp, _vp, _vp, _vp, _i, _i, _d, _i, _d, _d, _ll, _i, _i, _vp, _vp, _vp]),
    "costmodel_predict": (_i, [_i, _i, _vp, _i, _vp, _vp, _vp]),
    "costmodel_zscore_fit": (_i, [_i, _i, _vp, _vp, _vp, _vp]),
    "costmodel_zscore_apply": (_i, [_i, _i, _vp, _vp, _vp, _i, _vp, _vp]),
    "costmodel_error": (_i, [_i, _vp, _vp, _vp, _vp]),
    "costmodel_set_option": (_i, [_i, _i]),
    "costmodel_last_cuda_error": (_i, []),
    "costmodel_launch_count": (_ll, []),
}

_lib = _B._lib
for _name, (_res, _args) in SIGNATURES.items():
    try:
        _fn = getattr(_lib, _name)
    except AttributeError:
        raise ImportError("%s does not export %s" % (_B.LIB_PATH, _name))
    _fn.restype = _res
    _fn.argtypes = _args

_ptr = _B._ptr


def _check(status, where):
    if status != _B.DSLASH_OK:
        raise _B.DslashError(status, where)


def costmodel_param_count(f: int) -> int:
    return int(_lib.costmodel_param_count(int(f)))


def costmodel_weight_count(f: int) -> int:
    return int(_lib.costmodel_weight_count(int(f)))


def costmodel_train_smem_bytes(f: int, batch: int, cluster_size: int) -> int:
    return int(_lib.costmodel_train_smem_bytes(int(f), int(batch), int(cluster_size)))


def costmodel_train(f, n, x, y, uniforms, perms, epochs, batch, lr0, lr_step, lr_gamma, weight_decay, max_steps, n_models,
                    cluster_size, params_out, epoch_loss_out, stream) -> None:
    _check(_lib.costmodel_train(int(f), int(n), _ptr(x), _ptr(y), _ptr(uniforms), _ptr(perms), int(epochs), int(batch),
                                float(lr0), int(lr_step), float(lr_gamma), float(weight_decay), int(max_steps), int(n_models),
                                int(cluster_size), _ptr(params_out), _ptr(epoch_loss_out), _ptr(stream)), "costmodel_train")


def costmodel_train_status(*args) -> int:
    """costmodel_train returning the raw status instead of raising (error-path tests)."""
    (f, n, x, y, uniforms, perms, epochs, batch, lr0, lr_step, lr_gamma, weight_decay, max_steps, n_models, cluster_size,
     params_out, epoch_loss_out, stream) = args
    return int(_lib.costmodel_train(int(f), int(n), _ptr(x), _ptr(y), _ptr(uniforms), _ptr(perms), int(epochs), int(batch),
                                    float(lr0), int(lr_step), float(lr_gamma), float(weight_decay), int(max_steps),
                                    int(n_models), int(cluster_size), _ptr(params_out), _ptr(epoch_loss_out), _ptr(stream)))


def costmodel_predict(f, n, params, n_models, x, pred, stream) -> None:
    _check(_lib.costmodel_predict(int(f), int(n), _ptr(params), int(n_models), _ptr(x), _ptr(pred), _ptr(stream)),
           "costmodel_predict")


def costmodel_zscore_fit(n, cols, a, mean, std, stream) -> None:
    _check(_lib.costmodel_zscore_fit(int(n), int(cols), _ptr(a), _ptr(mean), _ptr(std), _ptr(stream)), "costmodel_zscore_fit")


def costmodel_zscore_apply(n, cols, a, mean, std, inverse, out, stream) -> None:
    _check(_lib.costmodel_zscore_apply(int(n), int(cols), _ptr(a), _ptr(mean), _ptr(std), int(inverse), _ptr(out), _ptr(stream)),
           "costmodel_zscore_apply")


def costmodel_error(n, pred, y, out, stream) -> None:
    _check(_lib.costmodel_error(int(n), _ptr(pred), _ptr(y), _ptr(out), _ptr(stream)), "costmodel_error")


COSTMODEL_OPT_THREADS = 1


def costmodel_set_option(option: int, value: int) -> None:
    _check(_lib.costmodel_set_option(int(option), int(value)), "costmodel_set_option")


def costmodel_last_cuda_error() -> int:
    return int(_lib.costmodel_last_cuda_error())


def costmodel_launch_count() -> int:
    return int(_lib.costmodel_launch_count())


# ------------------------------------------------------------------ torch plumbing: device buffers and copies only
class CostModel:
    """The protocol of PAPER.md:305-321 on the device: standardise (training rows' statistics), train, predict, NRMSE.
    Holds device tensors; every number is produced by a costmodel_* kernel."""

    PAPER = dict(epochs=150, batch=16, lr0=0.01, lr_step=30, lr_gamma=0.1, weight_decay=1e-4)

    def __init__(self, f: int, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2301_03636_b200 needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.f = int(f)
        self.device = torch.device(device)
        self.params = None
        self.n_models = 0
        self.x_mean = self.x_std = self.y_mean = self.y_std = None

    def _stream(self):
        return self.torch.cuda.current_stream().cuda_stream

    def _dev(self, a, dtype=None):
        import numpy as np
        t = self.torch.from_numpy(np.ascontiguousarray(a, dtype=dtype or np.float64))
        return t.to(self.device)

    def _empty(self, *shape):
        return self.torch.empty(shape, dtype=self.torch.float64, device=self.device)

    def fit_scaler(self, x_train, y_train):
        """Z-score statistics of the training rows (Reading R25).  x_train [n, F], y_train [n]: device float64 tensors."""
        n = x_train.shape[0]
        self.x_mean, self.x_std = self._empty(self.f), self._empty(self.f)
        self.y_mean, self.y_std = self._empty(1), self._empty(1)
        costmodel_zscore_fit(n, self.f, x_train.data_ptr(), self.x_mean.data_ptr(), self.x_std.data_ptr(), self._stream())
        costmodel_zscore_fit(n, 1, y_train.data_ptr(), self.y_mean.data_ptr(), self.y_std.data_ptr(), self._stream())

    def scale_x(self, x):
        out = self.torch.empty_like(x)
        costmodel_zscore_apply(x.shape[0], self.f, x.data_ptr(), self.x_mean.data_ptr(), self.x_std.data_ptr(), 0, out.data_ptr(),
                               self._stream())
        return out

    def scale_y(self, y, inverse=False):
        out = self.torch.empty_like(y)
        costmodel_zscore_apply(y.numel(), 1, y.data_ptr(), self.y_mean.data_ptr(), self.y_std.data_ptr(), int(inverse),
                               out.data_ptr(), self._stream())
        return out

    def train(self, xs, ys, uniforms, perms, epochs=150, batch=16, lr0=0.01, lr_step=30, lr_gamma=0.1, weight_decay=1e-4,
              max_steps=-1, cluster_size=0):
        """xs [n, F], ys [n] standardised device tensors; uniforms [n_models, weight_count] float64, perms
        [n_models, epochs, n] int32 (device tensors).  Returns (params [n_models, param_count], epoch_loss [n_models, epochs])."""
        n = xs.shape[0]
        n_models = uniforms.shape[0] if uniforms.dim() == 2 else 1
        self.n_models = n_models
        self.params = self._empty(n_models, costmodel_param_count(self.f))
        loss = self._empty(n_models, max(epochs, 1))
        costmodel_train(self.f, n, xs.data_ptr(), ys.data_ptr(), uniforms.data_ptr(), perms.data_ptr() if epochs > 0 else 0, epochs,
                        batch, lr0, lr_step, lr_gamma, weight_decay, max_steps, n_models, cluster_size, self.params.data_ptr(),
                        loss.data_ptr(), self._stream())
        return self.params, loss[:, :epochs]

    def predict(self, xs, params=None):
        """Standardised predictions [n_models, n] for standardised rows xs [n, F]."""
        params = self.params if params is None else params
        n_models = params.shape[0] if params.dim() == 2 else 1
        pred = self._empty(n_models, xs.shape[0])
        costmodel_predict(self.f, xs.shape[0], params.data_ptr(), n_models, xs.data_ptr(), pred.data_ptr(), self._stream())
        return pred

    def error(self, pred, y):
        """(RMSE, NRMSE) of one prediction vector against y (Eq. 2, Eq. 3), as a device tensor of two doubles."""
        out = self._empty(2)
        costmodel_error(y.numel(), pred.data_ptr(), y.data_ptr(), out.data_ptr(), self._stream())
        return out
