"""zkd_seed_fp64_static (include/zkd.h): the fp64 seed (S1) with its scratch in a static device array, for callers that must
not call cudaMalloc.  Its output is compared with the existing path's (zkd_seed_fp64) within the tolerances of
test_seed_fp64_vs_lapack, on consecutive calls that share the array (a different matrix, then a smaller N, then the first
matrix again: stale contents must not leak).  This file sorts last on purpose: the suite runs with pytest -x."""
from __future__ import annotations

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def zkd():
    import torch

    assert torch.cuda.is_available()
    import paper_2402_11868_b200 as z

    z.lib()
    return z


def _herm(seed, batch, N):
    rng = np.random.default_rng(seed)
    A = rng.uniform(-1, 1, (batch, N, N)) + 1j * rng.uniform(-1, 1, (batch, N, N))
    return (A + A.conj().transpose(0, 2, 1)) / 2


def _run(fn, A):
    import torch

    batch, N, _ = A.shape
    dA = torch.from_numpy(np.ascontiguousarray(A.astype(np.complex128).view(np.float64))).cuda()
    mu = torch.full((batch * N,), float("nan"), dtype=torch.float64, device="cuda")
    V = torch.full((batch * N * N * 2,), float("nan"), dtype=torch.float64, device="cuda")
    fn(N, batch, dA, mu, V)
    torch.cuda.synchronize()
    return mu.cpu().numpy().reshape(batch, N), V.cpu().numpy().view(np.complex128).reshape(batch, N, N)


def _check_against_existing(zkd, A):
    batch, N, _ = A.shape
    mu_s, V_s = _run(zkd.seed_fp64_static, A)
    mu_e, V_e = _run(zkd.seed_fp64, A)
    for b in range(batch):
        F = max(np.linalg.norm(A[b]), 1.0)
        assert np.all(np.isfinite(mu_s[b])) and np.all(np.isfinite(V_s[b]))
        assert np.all(np.diff(mu_s[b]) >= 0)
        # the existing path's answer, within the tolerance test_seed_fp64_vs_lapack gives either of them against LAPACK
        assert np.max(np.abs(mu_s[b] - mu_e[b])) <= 2 * 1e-12 * F * N
        assert np.max(np.abs(V_s[b].conj().T @ V_s[b] - np.eye(N))) <= 1e-13 * N
        assert np.max(np.abs(A[b] @ V_s[b] - V_s[b] * mu_s[b][None, :])) <= 1e-11 * F
        # same eigenvectors up to the phase of a column (the spectra of these random matrices have no clusters)
        ov = np.abs(np.sum(V_e[b].conj() * V_s[b], axis=0))
        assert np.max(np.abs(ov - 1.0)) <= 1e-9
        if N > 256:  # the existing path runs the same blocked kernel there: same columns, phases included
            assert np.max(np.abs(V_s[b] - V_e[b])) <= 1e-10
    return mu_s, V_s


def test_static_seed_matches_existing_path_on_consecutive_calls(zkd):
    A1 = _herm(901, 1, 300)
    A2 = _herm(902, 1, 300)
    A3 = _herm(903, 3, 77)
    first = _check_against_existing(zkd, A1)
    _check_against_existing(zkd, A2)  # second call in a row, other contents in the shared array
    _check_against_existing(zkd, A3)  # smaller, ragged N and a batch: the array still holds a 300 x 300 G
    again = _check_against_existing(zkd, A1)
    assert np.array_equal(first[0], again[0]) and np.array_equal(first[1], again[1])  # nothing left over from the calls between


@pytest.mark.parametrize("N,batch", [(1, 2), (2, 1), (16, 4), (64, 2), (200, 1), (512, 1)])
def test_static_seed_sizes_up_to_the_maximum(zkd, N, batch):
    A = _herm(1000 + N, batch, N)
    _check_against_existing(zkd, A)
    _check_against_existing(zkd, A[::-1].copy())


def test_static_seed_rejects_sizes_beyond_its_array(zkd):
    import torch

    N = zkd.SEED_STATIC_MAX_N + 1
    dA = torch.zeros(N * N * 2, dtype=torch.float64, device="cuda")
    mu = torch.full((N,), 7.0, dtype=torch.float64, device="cuda")
    V = torch.zeros(N * N * 2, dtype=torch.float64, device="cuda")
    with pytest.raises(zkd.ZkdError) as e:
        zkd.seed_fp64_static(N, 1, dA, mu, V)
    assert e.value.code == -8 and "static" in str(e.value)
    torch.cuda.synchronize()
    assert float(mu.min()) == 7.0  # nothing was launched
