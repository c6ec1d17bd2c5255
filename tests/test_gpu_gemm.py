"""DMMA GEMM engine vs torch.matmul (cuBLAS, complex128/float64) -- unit parity of the building
blocks of S1/S3/S4.  Sizes span several tiles and ragged tails."""
import json
import os

import pytest
import torch

from gpu_util import cm, lg, randc, randr

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def eng():
    from paper_2310_03341_b200 import binding
    e = binding.Eigh(1024)
    yield e
    e.close()


def rel(a, b):
    return (a - b).abs().max().item() / max(b.abs().max().item(), 1e-300)


@pytest.mark.parametrize("opA,opB", [("N", "N"), ("N", "C"), ("C", "N")])
@pytest.mark.parametrize("M,N,K,small", [(128, 64, 8, 0), (300, 200, 77, 0), (64, 64, 1000, 0), (257, 129, 64, 2),
                                         (1, 1, 1, 0), (515, 70, 131, 0)])
def test_zgemm_variants(eng, opA, opB, M, N, K, small):
    A = randc(M, K, 1) if opA == "N" else randc(K, M, 1)
    B = randc(K, N, 2) if opB == "N" else randc(N, K, 2)
    C = randc(M, N, 3)
    As, Bs, Cs = cm(A), cm(B), cm(C)
    opa = A if opA == "N" else A.conj().t()
    opb = B if opB == "N" else B.conj().t()
    ref = -0.5 * (opa @ opb) + 1.0 * C
    eng.zgemm(opA, opB, M, N, K, -0.5, As, A.shape[0], Bs, B.shape[0], 1.0, Cs, M, lower_only=small)
    torch.cuda.synchronize()
    assert rel(lg(Cs), ref) < 1e-13
    # beta = 0 must not read C (NaN-safe)
    Cs2 = torch.full_like(Cs, float("nan"))
    eng.zgemm(opA, opB, M, N, K, 1.0, As, A.shape[0], Bs, B.shape[0], 0.0, Cs2, M, lower_only=small)
    torch.cuda.synchronize()
    assert rel(lg(Cs2), opa @ opb) < 1e-13


@pytest.mark.parametrize("M,N,K,splitk", [(64, 64, 5000, 37), (64, 48, 333, 4), (200, 64, 1024, 3)])
def test_zgemm_splitk(eng, M, N, K, splitk):
    A, B, C = randc(K, M, 4), randc(K, N, 5), randc(M, N, 6)
    As, Bs, Cs = cm(A), cm(B), cm(C)
    ref = 2.0 * (A.conj().t() @ B) + 1.0 * C
    eng.zgemm("C", "N", M, N, K, 2.0, As, K, Bs, K, 1.0, Cs, M, splitk=splitk)
    torch.cuda.synchronize()
    assert rel(lg(Cs), ref) < 1e-13


@pytest.mark.parametrize("M,K", [(128, 64), (517, 64), (1000, 128)])
def test_zgemm_her2k_lower(eng, M, K):
    """C -= V W^H + W V^H on the lower tiles only: lower triangle (and every 64-aligned diagonal
    block) must be exact; tiles strictly above the diagonal must be untouched."""
    V, W = randc(M, K, 7), randc(M, K, 8)
    C = randc(M, M, 9)
    C = C + C.conj().t()
    Vs, Ws, Cs = cm(V), cm(W), cm(C)
    ref = C - V @ W.conj().t() - W @ V.conj().t()
    eng.zgemm("N", "C", M, M, K, -1.0, Vs, M, Ws, M, 1.0, Cs, M, K2=K, A2=Ws, lda2=M, B2=Vs, ldb2=M, lower_only=1)
    torch.cuda.synchronize()
    out = lg(Cs)
    low = torch.tril(torch.ones(M, M, device="cuda", dtype=torch.bool))
    assert rel(out[low], ref[low]) < 1e-13
    for d0 in range(0, M, 64):
        d1 = min(M, d0 + 64)
        assert rel(out[d0:d1, d0:d1], ref[d0:d1, d0:d1]) < 1e-13
    # a tile strictly above the diagonal is untouched
    if M >= 256:
        assert torch.equal(out[0:64, 192:256], C[0:64, 192:256])


@pytest.mark.parametrize("M,N,splitk", [(64, 64, 1), (130, 64, 1), (1000, 64, 3), (777, 40, 2)])
def test_zhemm_lower(eng, M, N, splitk):
    """X = Herm(A) B reading only the lower triangle and the 64-aligned diagonal blocks."""
    A = randc(M, M, 10)
    A = A + A.conj().t()
    B = randc(M, N, 11)
    ref = A @ B
    G = A.clone()
    up = torch.triu(torch.ones(M, M, device="cuda", dtype=torch.bool), 1)
    blk = torch.zeros(M, M, device="cuda", dtype=torch.bool)
    for d0 in range(0, M, 64):
        blk[d0:d0 + 64, d0:d0 + 64] = True
    G[up & ~blk] = float("nan")                     # must never be read
    Gs, Bs = cm(G), cm(B)
    Xs = torch.full((N, M), float("nan"), dtype=torch.complex128, device="cuda")
    eng.zhemm_lower(M, N, Gs, M, Bs, M, Xs, M, splitk=splitk)
    torch.cuda.synchronize()
    assert rel(lg(Xs), ref) < 1e-13


@pytest.mark.parametrize("M,N,K", [(128, 128, 16), (300, 260, 77), (1, 1, 1), (515, 129, 250), (64, 700, 3)])
def test_dgemm(eng, M, N, K):
    lda = M + (M & 1)
    ldb = K + (K & 1)
    A = randr(lda, K + 5, 12)
    B = randr(ldb, N, 13)
    idx = torch.randperm(K + 5)[:K].to(torch.int32).cuda()
    As, Bs = cm(A), cm(B)
    Cs = torch.full((N, M), float("nan"), dtype=torch.float64, device="cuda")
    eng.dgemm(M, N, K, As, lda, Bs, ldb, Cs, M, col_idx=idx)
    torch.cuda.synchronize()
    ref = A[:M, idx.long()] @ B[:K, :]
    assert rel(lg(Cs), ref) < 1e-13
    Cs2 = torch.full((N, M), float("nan"), dtype=torch.float64, device="cuda")
    eng.dgemm(M, N, K, As, lda, Bs, ldb, Cs2, M)
    torch.cuda.synchronize()
    assert rel(lg(Cs2), A[:M, :K] @ B[:K, :]) < 1e-13
