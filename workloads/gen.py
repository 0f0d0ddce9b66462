"""Seeded synthetic workloads with the shapes of BASELINE.json `configs[0..4]` (C1..C5).

The datasets these shapes come from (ISOLET, named in PAPER.md L197; MNIST- and UCI-HAR-shaped
sizes in BASELINE.json) are not available offline; these generators stand in for them
(recipe: DESIGN.md "Input recipe").  Nothing here encodes, compares or
classifies: arrays are drawn from numpy PCG64 streams keyed by (BASE_SEED, config, array
name) and handed, identical, to the oracle and to the CUDA path.
"""
from __future__ import annotations

import zlib

import ml_dtypes
import numpy as np

BASE_SEED = 26547


def rng_for(cfg: int, name: str) -> np.random.Generator:
    """Independent PCG64 stream per (config index, array name)."""
    ss = np.random.SeedSequence([BASE_SEED, int(cfg), zlib.crc32(name.encode())])
    return np.random.Generator(np.random.PCG64(ss))


# ----------------------------------------------------------------------------- layout helpers
def pack_bits_lsb(bits: np.ndarray, ld_words: int | None = None) -> np.ndarray:
    """[R][D] array of 0/1 -> [R][ld_words] uint32, element d in word d>>5 at bit d&31
    (LSB first), tail bits and padding words zero.  Interface layout of include/hdc.h."""
    bits = np.ascontiguousarray(bits, dtype=np.uint8)
    R, D = bits.shape
    W = (D + 31) // 32
    ld = W if ld_words is None else int(ld_words)
    assert ld >= W
    padded = np.zeros((R, ld * 32), dtype=np.uint8)
    padded[:, :D] = bits
    by = np.packbits(padded, axis=1, bitorder="little")          # [R][ld*4] bytes, LSB first
    return by.view("<u4").reshape(R, ld).copy()


def to_bf16_bits(x: np.ndarray) -> np.ndarray:
    """float array -> uint16 bfloat16 bit patterns (library conversion, ml_dtypes)."""
    return np.asarray(x, dtype=np.float32).astype(ml_dtypes.bfloat16).view(np.uint16)


def from_bf16_bits(u: np.ndarray) -> np.ndarray:
    """uint16 bfloat16 bit patterns -> float32 (exact)."""
    return np.asarray(u, dtype=np.uint16).view(ml_dtypes.bfloat16).astype(np.float32)


def tile_rows(a: np.ndarray, n: int) -> np.ndarray:
    """Repeat the rows of `a` cyclically up to n rows (steady-state throughput inputs)."""
    reps = -(-n // a.shape[0])
    return np.ascontiguousarray(np.concatenate([a] * reps, axis=0)[:n])


# ----------------------------------------------------------------------------- tables
def id_table(cfg: int, F: int, D: int) -> np.ndarray:
    """[F][D] iid uniform bits (ID hypervectors)."""
    return rng_for(cfg, "id_bits").integers(0, 2, size=(F, D), dtype=np.uint8)


def level_table(cfg: int, Q: int, D: int) -> np.ndarray:
    """[Q][D] level hypervectors (reading A13): LV_0 iid random; LV_q = LV_0 with the first
    floor(q*(D/2)/(Q-1)) entries of one fixed random permutation flipped."""
    r = rng_for(cfg, "level_bits")
    lv0 = r.integers(0, 2, size=D, dtype=np.uint8)
    perm = r.permutation(D)
    out = np.empty((Q, D), dtype=np.uint8)
    for q in range(Q):
        m = 0 if Q == 1 else (q * (D // 2)) // (Q - 1)
        v = lv0.copy()
        v[perm[:m]] ^= 1
        out[q] = v
    return out


# ----------------------------------------------------------------------------- C1
def c1_tiny(D: int = 2048):
    """configs[0]: N=256/256, F=64 fp32 in [0,1] around K=4 centroids (sigma 0.1), P in {+-1}."""
    cfg, K, F, n_tr, n_te = 1, 4, 64, 256, 256
    mu = rng_for(cfg, "centroids").uniform(0.0, 1.0, size=(K, F))

    def split(name, n):
        y = (np.arange(n) % K).astype(np.int32)
        x = mu[y] + 0.1 * rng_for(cfg, name).standard_normal((n, F))
        return np.clip(x, 0.0, 1.0).astype(np.float32), y

    Xtr, ytr = split("x_train", n_tr)
    Xte, yte = split("x_test", n_te)
    P = (1.0 - 2.0 * rng_for(cfg, "proj").integers(0, 2, size=(D, F))).astype(np.float32)
    return dict(name="C1", K=K, F=F, D=D, Xtr=Xtr, ytr=ytr, Xte=Xte, yte=yte, P=P)


# ----------------------------------------------------------------------------- C2 / C4
def _gaussian_mixture(cfg, K, F, sigma, n_tr, n_te, D):
    g = rng_for(cfg, "centroids").standard_normal((K, F))
    mu = g / np.linalg.norm(g, axis=1, keepdims=True)

    def split(name, n):
        y = rng_for(cfg, name + "_y").integers(0, K, size=n).astype(np.int32)
        x = mu[y] + sigma * rng_for(cfg, name).standard_normal((n, F))
        return x.astype(np.float32), y

    Xtr, ytr = split("x_train", n_tr)
    Xte, yte = split("x_test", n_te)
    # generated once at full D, independently per row d => prefix-stable under D_eff (S3)
    P = rng_for(cfg, "proj").standard_normal((D, F)).astype(np.float32)
    return Xtr, ytr, Xte, yte, P


def c2_isolet_shaped(D: int = 10000, n_tr: int = 6238, n_te: int = 1559):
    """configs[1]: F=617, K=26 Gaussian mixture (unit-norm centroids, sigma 0.3), Gaussian P."""
    Xtr, ytr, Xte, yte, P = _gaussian_mixture(2, 26, 617, 0.3, n_tr, n_te, D)
    return dict(name="C2", K=26, F=617, D=D, Xtr=Xtr, ytr=ytr, Xte=Xte, yte=yte, P=P,
                epochs=20, lr=0.05)


def c4_har_shaped(D: int = 10000, n_tr: int = 7352, n_te: int = 2947):
    """configs[3]: F=561, K=6 Gaussian mixture (sigma 0.4); P generated once at D=10000."""
    Xtr, ytr, Xte, yte, P = _gaussian_mixture(4, 6, 561, 0.4, n_tr, n_te, D)
    return dict(name="C4", K=6, F=561, D=D, Xtr=Xtr, ytr=ytr, Xte=Xte, yte=yte, P=P,
                d_eff=(10000, 8192, 4096, 2048, 1024), epochs=(0, 5, 20), lr=0.05)


# ----------------------------------------------------------------------------- C3
def c3_mnist_shaped(D: int = 10000, n_tr: int = 60000, n_te: int = 10000, Q: int = 256):
    """configs[2]: 28x28 uint8 images, ~80% zeros, class-dependent Gaussian blob patterns,
    K=10; level index = pixel value (Q=256); ID and level tables as packed-bit inputs."""
    cfg, K, side = 3, 10, 28
    F = side * side
    r = rng_for(cfg, "class_blobs")
    blobs = []
    for _ in range(K):
        nb = int(r.integers(3, 6))
        blobs.append(dict(c=r.uniform(5.0, 23.0, size=(nb, 2)), s=r.uniform(1.6, 2.8, size=nb),
                          a=r.uniform(0.7, 1.0, size=nb)))
    yy, xx = np.meshgrid(np.arange(side, dtype=np.float64), np.arange(side, dtype=np.float64),
                         indexing="ij")

    def split(name, n):
        rr = rng_for(cfg, name)
        y = rr.integers(0, K, size=n).astype(np.int32)
        img = np.zeros((n, side, side), dtype=np.float64)
        for k in range(K):
            idx = np.nonzero(y == k)[0]
            if idx.size == 0:
                continue
            b = blobs[k]
            for j in range(b["s"].size):
                cj = b["c"][j] + 1.5 * rr.standard_normal((idx.size, 2))
                aj = b["a"][j] * rr.uniform(0.8, 1.2, size=idx.size)
                r2 = (yy[None] - cj[:, 0, None, None]) ** 2 + (xx[None] - cj[:, 1, None, None]) ** 2
                img[idx] += aj[:, None, None] * np.exp(-r2 / (2.0 * b["s"][j] ** 2))
        img = np.minimum(1.0, img)
        img[img < 0.20] = 0.0
        return np.rint(255.0 * img).astype(np.uint8).reshape(n, F), y

    Ltr, ytr = split("x_train", n_tr)
    Lte, yte = split("x_test", n_te)
    return dict(name="C3", K=K, F=F, D=D, Q=Q, Ltr=Ltr, ytr=ytr, Lte=Lte, yte=yte,
                ID=id_table(cfg, F, D), LV=level_table(cfg, Q, D))


# ----------------------------------------------------------------------------- C5
def c5_large_batch(n: int, batch: int = 0, D: int = 16384, K: int = 1000, F: int = 1024,
                   n_unstructured: int = 0, per_class: int = 32):
    """configs[4]: F=1024 bf16 features ~N(0,1) around K=1000 centroids, P~N(0,1) in bf16.

    Returns `n` structured queries of device batch `batch` (x=(M_y+eps)/sqrt2), optionally
    followed by `n_unstructured` queries x~N(0,I) whose scores sit near zero (tie stress),
    plus `per_class` noisy training samples per class from which either side bundles its own
    class hypervectors.  All float arrays are exactly bf16-representable float32.
    """
    cfg = 5
    M = rng_for(cfg, "centroids").standard_normal((K, F))
    rq = rng_for(cfg, f"x_batch{batch}")
    y = rq.integers(0, K, size=n).astype(np.int32)
    X = (M[y] + rq.standard_normal((n, F))) / np.sqrt(2.0)
    if n_unstructured:
        X = np.concatenate([X, rng_for(cfg, f"x_unstructured{batch}").standard_normal(
            (n_unstructured, F))], axis=0)
        y = np.concatenate([y, np.full(n_unstructured, -1, dtype=np.int32)])
    rt = rng_for(cfg, "x_train")
    ytr = np.repeat(np.arange(K, dtype=np.int32), per_class)
    Xtr = (M[ytr] + rt.standard_normal((ytr.size, F))) / np.sqrt(2.0)
    P = rng_for(cfg, "proj").standard_normal((D, F))
    q = lambda a: from_bf16_bits(to_bf16_bits(a))                      # noqa: E731
    return dict(name="C5", K=K, F=F, D=D, X=q(X), y=y, Xtr=q(Xtr), ytr=ytr, P=q(P))
