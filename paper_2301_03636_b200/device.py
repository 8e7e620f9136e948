"""Device-side plumbing around the C ABI: torch owns device memory and streams, nothing else.

`Lattice` wraps one dslash_ctx plus the handful of copies a caller needs to get canonical NumPy
fields to the device in the ctx's native layout and back.  All arithmetic and all layout
conversion happen in libdslash_b200.so (dslash_pack_* / dslash_apply / dslash_unpack_spinor).
"""
import numpy as np
import torch

from . import binding as B

PRECISIONS = {"f64": B.DSLASH_FP64, "f32": B.DSLASH_FP32}
LAYOUTS = {"aos": B.DSLASH_AOS, "soa": B.DSLASH_SOA}


class Lattice:
    def __init__(self, dims, precision="f64", layout="soa", recon12=False, device="cuda:0"):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2301_03636_b200 needs a CUDA device; there is no CPU fallback")
        self.dims = tuple(int(d) for d in dims)
        self.volume = int(np.prod(self.dims))
        self.precision, self.layout, self.recon12 = precision, layout, bool(recon12)
        self.np_dtype = np.float64 if precision == "f64" else np.float32
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.ctx = B.dslash_create(self.dims, PRECISIONS[precision], LAYOUTS[layout] | (B.DSLASH_RECON12 if recon12 else 0))

    # -- lifetime
    def close(self):
        if getattr(self, "ctx", None):
            B.dslash_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass

    # -- memory
    @staticmethod
    def stream():
        return torch.cuda.current_stream().cuda_stream

    def _bytes(self, n):
        return torch.empty(int(n), dtype=torch.uint8, device=self.device)

    def new_spinor(self):
        return self._bytes(B.dslash_spinor_bytes(self.ctx))

    def new_gauge(self):
        return self._bytes(B.dslash_gauge_bytes(self.ctx))

    def _to_device(self, a):
        a = np.ascontiguousarray(a, dtype=self.np_dtype)
        return torch.from_numpy(a.reshape(-1).view(np.uint8)).to(self.device)

    def upload_spinor(self, canonical):
        """canonical NumPy spinor [T,Z,Y,X,4,3,2] -> native device buffer."""
        assert canonical.size == self.volume * 24
        src = self._to_device(canonical)
        dst = self.new_spinor()
        B.dslash_pack_spinor(self.ctx, dst.data_ptr(), src.data_ptr(), self.stream())
        torch.cuda.current_stream().synchronize()
        return dst

    def upload_gauge(self, canonical):
        """canonical NumPy gauge [T,Z,Y,X,4,3,3,2] (18 reals per link) -> native device buffer."""
        assert canonical.size == self.volume * 72
        src = self._to_device(canonical)
        dst = self.new_gauge()
        B.dslash_pack_gauge(self.ctx, dst.data_ptr(), src.data_ptr(), self.stream())
        torch.cuda.current_stream().synchronize()
        return dst

    def download_spinor(self, native):
        """native device spinor -> canonical NumPy [T,Z,Y,X,4,3,2] at the ctx's precision."""
        dst = self._bytes(B.dslash_canonical_spinor_bytes(self.ctx))
        B.dslash_unpack_spinor(self.ctx, dst.data_ptr(), native.data_ptr(), self.stream())
        lx, ly, lz, lt = self.dims
        return dst.cpu().numpy().view(self.np_dtype).reshape(lt, lz, ly, lx, 4, 3, 2)

    # -- the operator
    def apply(self, out, inp, gauge):
        B.dslash_apply(self.ctx, out.data_ptr(), inp.data_ptr(), gauge.data_ptr(), self.stream())

    def tune(self, out, inp, gauge):
        """dslash_tune: time the eligible kernels on these buffers and keep the fastest; returns (kernel, ms)."""
        return B.dslash_tune(self.ctx, out.data_ptr(), inp.data_ptr(), gauge.data_ptr(), self.stream())

    def apply_op(self, op, mass, out, inp, gauge):
        B.dslash_apply_op(self.ctx, op, mass, out.data_ptr(), inp.data_ptr(), gauge.data_ptr(), self.stream())

    def cg_solve(self, x, b, gauge, mass, tol, max_iter):
        """x <- solution of M^dagger M x = b (native device buffers); returns (iterations, rel_residual)."""
        return B.dslash_cg_solve(self.ctx, x.data_ptr(), b.data_ptr(), gauge.data_ptr(), mass, tol, max_iter, self.stream())

    # -- even-odd (checkerboarded) form; all extents even
    def new_eo_spinor(self):
        return self._bytes(B.dslash_eo_spinor_bytes(self.ctx)).zero_()

    def upload_eo_spinor(self, canonical, parity):
        """canonical full-lattice NumPy spinor -> native half-lattice device buffer holding its sites of `parity`."""
        assert canonical.size == self.volume * 24
        src = self._to_device(canonical)
        dst = self.new_eo_spinor()
        B.dslash_eo_pack_spinor(self.ctx, dst.data_ptr(), src.data_ptr(), parity, self.stream())
        torch.cuda.current_stream().synchronize()
        return dst

    def upload_eo_gauge(self, canonical):
        assert canonical.size == self.volume * 72
        src = self._to_device(canonical)
        dst = self._bytes(B.dslash_eo_gauge_bytes(self.ctx))
        B.dslash_eo_pack_gauge(self.ctx, dst.data_ptr(), src.data_ptr(), self.stream())
        torch.cuda.current_stream().synchronize()
        return dst

    def download_eo_spinor(self, halves):
        """{parity: native half-lattice buffer} -> canonical full-lattice NumPy spinor (absent parities are zero)."""
        dst = self._bytes(B.dslash_canonical_spinor_bytes(self.ctx)).zero_()
        for parity, buf in halves.items():
            B.dslash_eo_unpack_spinor(self.ctx, dst.data_ptr(), buf.data_ptr(), parity, self.stream())
        lx, ly, lz, lt = self.dims
        return dst.cpu().numpy().view(self.np_dtype).reshape(lt, lz, ly, lx, 4, 3, 2)

    def eo_apply(self, out_parity, dagger, out, inp, gauge_eo):
        B.dslash_eo_apply(self.ctx, out_parity, dagger, out.data_ptr(), inp.data_ptr(), gauge_eo.data_ptr(), self.stream())

    def eo_apply_schur(self, dagger, mass, out_even, in_even, tmp_odd, gauge_eo):
        B.dslash_eo_apply_schur(self.ctx, dagger, mass, out_even.data_ptr(), in_even.data_ptr(), tmp_odd.data_ptr(),
                                gauge_eo.data_ptr(), self.stream())

    def eo_apply_schur_static(self, dagger, mass, out_even, in_even, gauge_eo):
        """The same operator with the intermediate in the library's built-in array: nothing is allocated (half-lattice
        fields up to B.DSLASH_STATIC_SCRATCH_BYTES; calls that overlap on the GPU share that array)."""
        B.dslash_eo_apply_schur_static(self.ctx, dagger, mass, out_even.data_ptr(), in_even.data_ptr(), gauge_eo.data_ptr(),
                                       self.stream())

    def eo_cg_solve(self, x_even, b_even, gauge_eo, mass, tol, max_iter):
        """x_even <- solution of Mhat^dagger Mhat x = b_even; returns (iterations, rel_residual)."""
        return B.dslash_eo_cg_solve(self.ctx, x_even.data_ptr(), b_even.data_ptr(), gauge_eo.data_ptr(), mass, tol, max_iter,
                                    self.stream())

    def eo_solve(self, x_even, x_odd, b_even, b_odd, gauge_eo, mass, tol, max_iter):
        """(x_even, x_odd) <- solution of M x = b through the even-odd preconditioned system."""
        return B.dslash_eo_solve(self.ctx, x_even.data_ptr(), x_odd.data_ptr(), b_even.data_ptr(), b_odd.data_ptr(),
                                 gauge_eo.data_ptr(), mass, tol, max_iter, self.stream())

    def set_variant(self, depth, tpb=0, spt=0):
        B.dslash_set_variant(self.ctx, depth, tpb, spt)

    def set_tile(self, tile):
        B.dslash_set_tile(self.ctx, tile)

    def set_kernel(self, kernel):
        B.dslash_set_kernel(self.ctx, {"auto": B.DSLASH_KERNEL_AUTO, "direct": B.DSLASH_KERNEL_DIRECT,
                                       "wpipe": B.DSLASH_KERNEL_WARP_PIPE, "march": B.DSLASH_KERNEL_MARCH}.get(kernel, kernel))

    def dslash(self, gauge_canonical, spinor_canonical):
        """Convenience: canonical NumPy in -> canonical NumPy out (one application on the device)."""
        g = self.upload_gauge(gauge_canonical)
        p = self.upload_spinor(spinor_canonical)
        o = self.new_spinor()
        self.apply(o, p, g)
        return self.download_spinor(o)
