#!/usr/bin/env python
"""Writes tests/golden/config3_full_oracle.npz: the fp64 CPU oracle's H p0 and H^T y on BASELINE config 3 at
its FULL length (256^3, 2000 samples, 2048 receivers), reduced to what a test can carry in the repository.

Calls only oracle/ and the seeded input generators (paper_1709_02733_b200/synth.py, which holds none of the
method's arithmetic).  The CUDA path is never imported.  Takes about half an hour on 8 cores
(2 x 3.4e10 cell updates).  Run:  python tests/golden/make_config3_golden.py

What is stored ("full-length oracle runs for C1, C2, C3"; the GPU suite has 20 minutes in all, so
this run cannot be repeated inside it):
  inputs   p0 = config 3's own p0 ; y = standard normal (nt x L) from default_rng(Y_SEED), cast to fp32
  data     rows of H p0 for every 32nd receiver (fp64) ; K random-sign sums over all receivers per time sample
           and their l2 norms (a sum is linear in the error, so a wrong receiver shows at first order)
  image    three full-resolution planes of H^T y through the grid centre (fp64 -> fp32 storage) ; for every
           (32 x 32 tile, z plane) K random-sign sums and the l2 norm, so that no brick of the fused kernel's
           decomposition can hide an error in the 1.7e7-cell norm
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

Y_SEED = 330
SIGN_SEED = 331
K = 2
RCV_STRIDE = 32
TILE = 32
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config3_full_oracle.npz")


def signs(shape):
    """K seeded +-1 arrays of the given shape (int8)."""
    rng = np.random.default_rng(SIGN_SEED)
    return (rng.integers(0, 2, size=(K,) + tuple(shape), dtype=np.int8) * 2 - 1).astype(np.int8)


def reduce_data(d):
    d = np.asarray(d, dtype=np.float64)
    s = signs((d.shape[1],)).astype(np.float64)                 # [K][L]
    return dict(data_rows=d[:, ::RCV_STRIDE].copy(), data_sums=d @ s.T, data_norms=np.linalg.norm(d, axis=1))


def reduce_image(img):
    img = np.asarray(img, dtype=np.float64)
    nz, ny, nx = img.shape
    s = signs((ny, nx)).astype(np.float64)                       # [K][ny][nx], the same pattern on every plane
    ty, tx = ny // TILE, nx // TILE
    blk = img.reshape(nz, ty, TILE, tx, TILE)
    sums = np.stack([(blk * s[k].reshape(1, ty, TILE, tx, TILE)).sum(axis=(2, 4)) for k in range(K)])   # [K][nz][ty][tx]
    norms = np.sqrt((blk * blk).sum(axis=(2, 4)))
    return dict(image_plane_z=img[nz // 2].astype(np.float32), image_plane_y=img[:, ny // 2].astype(np.float32),
                image_plane_x=img[:, :, nx // 2].astype(np.float32), image_tile_sums=sums, image_tile_norms=norms,
                image_l2=np.float64(np.linalg.norm(img)), image_absmax=np.float64(np.abs(img).max()))


def adjoint_input(nt, L):
    return np.random.default_rng(Y_SEED).standard_normal((nt, L)).astype(np.float32)


def main():
    from paper_1709_02733_b200 import synth
    from oracle.oracle import Oracle, threads
    prob = synth.make_config(3)
    o = Oracle.from_problem(prob)
    print(f"config 3: {prob.prm.nx}^3, nt={prob.prm.nt}, L={prob.L}; oracle threads {threads()}", flush=True)
    t = time.time()
    d = o.forward(prob.p0.astype(np.float32).astype(np.float64))
    print(f"forward {time.time() - t:.0f} s", flush=True)
    t = time.time()
    img = o.adjoint(adjoint_input(prob.prm.nt, prob.L).astype(np.float64))
    print(f"adjoint {time.time() - t:.0f} s", flush=True)
    o.close()
    rec = dict(y_seed=np.int64(Y_SEED), sign_seed=np.int64(SIGN_SEED), rcv_stride=np.int64(RCV_STRIDE),
               data_l2=np.float64(np.linalg.norm(d)), data_absmax=np.float64(np.abs(d).max()))
    rec.update(reduce_data(d))
    rec.update(reduce_image(img))
    np.savez_compressed(OUT, **rec)
    print("wrote", OUT, os.path.getsize(OUT), "bytes")


if __name__ == "__main__":
    main()
