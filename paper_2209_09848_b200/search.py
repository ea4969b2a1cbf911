"""Convenience wrapper: allocates the output tensors with torch and calls the C ABI."""
from __future__ import annotations

from typing import Optional, Tuple

import numpy as np

from . import binding as B


class MatchedFilter:
    """One library context bound to the current torch CUDA stream of `device`."""

    def __init__(self, device: int = 0, topk: int = 0, snr_threshold: float = float("-inf"),
                 force_generic: bool = False, record_events: bool = False, workspace_limit_mb: int = 0,
                 shift_stack: bool = False, filter: int = 0, prf_table=None, sep_shape: int = 0):
        """filter: tno_mf_config::filter (0 Gaussian PRF, 1 shift-stack, 2 pixel-integrated Gaussian, 3 tabulated:
        prf_table [n_phase, 5], 4 tabulated non-separable: prf_table [n_phase_y, n_phase_x, 5, 5])."""
        import torch
        self._torch = torch
        self.device = torch.device("cuda", device)
        self.topk = int(topk)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        self.ctx = B.tno_mf_create(device, stream, topk, snr_threshold, force_generic, record_events,
                                   workspace_limit_mb, shift_stack, filter, sep_shape)
        if prf_table is not None:
            if int(filter) == 4:
                B.tno_mf_set_prf_table2d(self.ctx, prf_table)
            else:
                B.tno_mf_set_prf_table(self.ctx, prf_table)

    def close(self) -> None:
        if self.ctx is not None:
            self._torch.cuda.synchronize(self.device)
            B.tno_mf_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def search(self, frames, sigma_t, trajectories, prf_sigma: float, t0: float,
               want_maps: bool = True, out_snr=None, out_topk=None, frame_times=None, jitter_xy=None,
               valid=None):
        """Returns (snr maps tensor [n, H, W] or None, candidate tensor or None); asynchronous.
        frame_times [T] / jitter_xy [T, 2] (host, optional) go through tno_mf_search_ex; valid (CUDA
        tensor shaped like frames, optional) through tno_mf_search_masked."""
        torch = self._torch
        n = np.asarray(trajectories).shape[0]
        T, H, W = frames.shape
        if want_maps and out_snr is None:
            out_snr = torch.empty((n, H, W), dtype=torch.float32, device=frames.device)
        if self.topk > 0 and out_topk is None:
            out_topk = torch.empty((n, self.topk, 4), dtype=torch.int32, device=frames.device)
        if valid is not None:
            B.tno_mf_search_masked(self.ctx, frames, valid, sigma_t, frame_times, jitter_xy, trajectories,
                                   prf_sigma, t0, out_snr if want_maps else None,
                                   out_topk if self.topk > 0 else None)
        elif frame_times is None and jitter_xy is None:
            B.tno_mf_search(self.ctx, frames, sigma_t, trajectories, prf_sigma, t0,
                            out_snr if want_maps else None, out_topk if self.topk > 0 else None)
        else:
            B.tno_mf_search_ex(self.ctx, frames, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma, t0,
                               out_snr if want_maps else None, out_topk if self.topk > 0 else None)
        return (out_snr if want_maps else None), (out_topk if self.topk > 0 else None)

    def search_max(self, frames, sigma_t, trajectories, prf_sigma: float, t0: float, want_maps: bool = False,
                   frame_times=None, jitter_xy=None, valid=None):
        """The search with the max over the bank fused in: (max map [H, W], arg-max trajectory
        [H, W], snr maps or None, candidate tensor or None); asynchronous."""
        torch = self._torch
        n = np.asarray(trajectories).shape[0]
        T, H, W = frames.shape
        mx = torch.empty((H, W), dtype=torch.float32, device=frames.device)
        ak = torch.empty((H, W), dtype=torch.int32, device=frames.device)
        snr = torch.empty((n, H, W), dtype=torch.float32, device=frames.device) if want_maps else None
        top = torch.empty((n, self.topk, 4), dtype=torch.int32, device=frames.device) if self.topk > 0 else None
        B.tno_mf_search_max(self.ctx, frames, valid, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma, t0,
                            mx, ak, snr, top)
        return mx, ak, snr, top

    def search_host(self, frames_host, sigma_t, trajectories, prf_sigma: float, t0: float, out_snr_host=None,
                    out_topk_host=None, frame_times=None, jitter_xy=None) -> None:
        """Stack and outputs in HOST memory (torch CPU tensors, pinned for overlap, or numpy arrays); the
        upload is overlapped with the search.  Returns when the results are in the host buffers."""
        B.tno_mf_search_host(self.ctx, frames_host, sigma_t, frame_times, jitter_xy, trajectories, prf_sigma, t0,
                             out_snr_host, out_topk_host)

    def background(self, frames, jitter_xy, delta: float, n_iter: int, in_place: bool = False):
        """PAPER.md section 3.1 on a stack with the scattered light removed: (coefficients [6, H, W], residual
        stack [T, H, W] -- `frames` itself if in_place)."""
        coef = self._torch.empty((6,) + tuple(frames.shape[1:]), dtype=self._torch.float32, device=frames.device)
        res = frames if in_place else self._torch.empty_like(frames)
        B.tno_mf_background(self.ctx, frames, jitter_xy, delta, n_iter, coef, res)
        return coef, res

    def flux(self, snr):
        """Flux estimate N / D of the maps of the last search on this context."""
        out = self._torch.empty_like(snr)
        B.tno_mf_flux(self.ctx, snr, out)
        return out

    def best(self, snr, box: int = 255):
        """PAPER.md section 3.3 on SNR maps [n, H, W]: (max over trajectories, arg-max trajectory, Z =
        max / local sigma of the box, top-K records of Z or None); asynchronous."""
        torch = self._torch
        n, H, W = snr.shape
        mx = torch.empty((H, W), dtype=torch.float32, device=snr.device)
        ak = torch.empty((H, W), dtype=torch.int32, device=snr.device)
        z = torch.empty((H, W), dtype=torch.float32, device=snr.device)
        top = torch.empty((self.topk, 4), dtype=torch.int32, device=snr.device) if self.topk > 0 else None
        B.tno_mf_best(self.ctx, snr, box, mx, ak, z, top)
        return mx, ak, z, top

    def peaks(self, score, radius: int, argk=None):
        """Non-maximum suppression of a score map [H, W] (e.g. Z of best()): (map with the score at the peaks and
        -inf elsewhere, top-K records of the peaks or None); asynchronous."""
        torch = self._torch
        out = torch.empty_like(score)
        top = torch.empty((self.topk, 4), dtype=torch.int32, device=score.device) if self.topk > 0 else None
        B.tno_mf_peaks(self.ctx, score, argk, radius, out, top)
        return out, top

    def inject(self, frames, trajs, xs, ys, amps, prf_sigma: float, t0: float, frame_times=None,
               jitter_xy=None) -> None:
        B.tno_mf_inject_ex(self.ctx, frames, frame_times, jitter_xy, B.make_sources(trajs, xs, ys, amps), prf_sigma, t0)

    @staticmethod
    def candidates_to_numpy(out_topk) -> np.ndarray:
        """[n, topk] structured array (snr, x, y, k) from the int32 [n, topk, 4] device tensor."""
        a = out_topk.cpu().numpy()
        return a.view(B.CAND_DTYPE).reshape(a.shape[0], a.shape[1])

    def stats(self) -> Tuple[int, int]:
        return B.tno_mf_last_stats(self.ctx)

    def kernel_ms(self) -> float:
        return B.tno_mf_last_kernel_ms(self.ctx)

    def work(self) -> Tuple[float, float, float]:
        return B.tno_mf_last_work(self.ctx)
