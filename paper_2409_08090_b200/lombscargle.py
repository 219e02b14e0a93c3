"""Astropy-style front end (the paper's user-facing surface is Astropy's LombScargle with
method="fastnifty").  Argument marshalling only: the frequency grid rule and buffer handling live
here, every arithmetic step of the periodogram runs in libls_b200.so.

    ls = LombScargle(t, y, dy, fit_mean=True, normalization="standard")
    freq, power = ls.autopower(samples_per_peak=5, nyquist_factor=5)        # Astropy's default grid heuristic
    power = ls.power_grid(f0, df, Nf)                                       # explicit regular grid

t: [Nd]; y: [Nd] or [batch, Nd]; dy: scalar, [Nd] or [batch, Nd] (numpy arrays or torch CUDA tensors).  Results are
torch CUDA tensors.  The NUFFT method needs a REGULAR frequency grid (Eq. 1: f_k = f0 + k df).
"""
from __future__ import annotations

import numpy as np

from . import binding as B

_NORM = {"standard": B.LS_NORM_STANDARD, "model": B.LS_NORM_MODEL, "log": B.LS_NORM_LOG, "psd": B.LS_NORM_PSD}


class LombScargle:
    def __init__(self, t, y, dy=None, fit_mean=True, normalization="standard", eps=None, dtype="float64", device=0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("LombScargle needs a CUDA device: the library has no CPU fallback")
        if normalization not in _NORM:
            raise ValueError(f"normalization must be one of {sorted(_NORM)}")
        if dtype not in ("float64", "float32"):
            raise ValueError("dtype must be 'float64' or 'float32'")
        self._torch = torch
        self.device = torch.device("cuda", device)
        self.fit_mean, self.normalization = bool(fit_mean), normalization
        self._tdt = torch.float64 if dtype == "float64" else torch.float32
        self.eps = float(eps) if eps is not None else (1e-9 if dtype == "float64" else 1e-5)

        def dev(a, dt):
            a = a if torch.is_tensor(a) else torch.as_tensor(np.asarray(a))
            return a.to(device=self.device, dtype=dt).contiguous()

        self.t = dev(t, torch.float64)                           # times always fp64 (reading A9)
        if self.t.ndim != 1 or self.t.numel() < 1:
            raise ValueError("t must be one-dimensional")
        y = dev(y, self._tdt)
        self.y = y[None] if y.ndim == 1 else y
        if self.y.ndim != 2 or self.y.shape[1] != self.t.numel():
            raise ValueError("y must be [Nd] or [batch, Nd]")
        if dy is None:
            dy = 1.0
        dy = dev(dy, self._tdt)
        if dy.ndim == 0:
            dy = dy.expand(self.t.numel()).contiguous()
        if dy.shape not in (self.t.shape, self.y.shape):
            raise ValueError("dy must be a scalar, [Nd] or [batch, Nd]")
        self.dy = dy
        self._plans = {}

    # ------------------------------------------------------------------ grids
    def autofrequency(self, samples_per_peak=5, nyquist_factor=5, minimum_frequency=None, maximum_frequency=None):
        """(f0, df, Nf) of Astropy's heuristic: df = 1/(samples_per_peak T), f0 = df/2 unless given, up to
        nyquist_factor times the average Nyquist frequency unless maximum_frequency is given."""
        T = float(self.t.max() - self.t.min())
        df = 1.0 / (samples_per_peak * T)
        f0 = 0.5 * df if minimum_frequency is None else float(minimum_frequency)
        fmax = 0.5 * nyquist_factor * self.t.numel() / T if maximum_frequency is None else float(maximum_frequency)
        return f0, df, max(1, int(round((fmax - f0) / df)))

    # ------------------------------------------------------------------ power
    def power_grid(self, f0, df, Nf, stream=None):
        """Power [batch, Nf] (or [Nf] for a single series) at f0 + k df, k = 0..Nf-1."""
        torch = self._torch
        batch, per = self.y.shape[0], self.dy.ndim == 2
        key = (float(f0), float(df), int(Nf))
        plan = self._plans.get(key)
        if plan is None:
            plan = B.Plan(self.t.numel(), int(Nf), float(f0), float(df), self.eps,
                          B.LS_F64 if self._tdt == torch.float64 else B.LS_F32, batch, dy_per_series=int(per),
                          no_floating_mean=0 if self.fit_mean else 1, normalization=_NORM[self.normalization],
                          device=self.device.index or 0)
            self._plans = {key: plan}                            # one cached plan: a new grid replaces it
        P = torch.empty((batch, int(Nf)), dtype=self._tdt, device=self.device)
        s = torch.cuda.current_stream(self.device) if stream is None else stream
        plan.execute(self.t, self.y, self.dy, P, s.cuda_stream)
        return P[0] if batch == 1 else P

    def autopower(self, **kw):
        f0, df, Nf = self.autofrequency(**kw)
        freq = f0 + df * self._torch.arange(Nf, dtype=self._torch.float64, device=self.device)
        return freq, self.power_grid(f0, df, Nf)

    def close(self):
        for p in self._plans.values():
            p.close()
        self._plans = {}
