"""Helpers for the -m gpu tests: column-major marshalling between torch and the C ABI."""
import torch


def cm(A):
    """Logical (M, K) tensor -> storage tensor (K, M) row-major == A column-major with ld = M."""
    return A.t().contiguous()


def lg(S):
    """Inverse of cm(): storage (K, M) -> logical (M, K) view."""
    return S.t()


def randc(m, n, seed, device="cuda"):
    g = torch.Generator(device="cpu").manual_seed(seed)
    a = torch.randn(m, n, dtype=torch.float64, generator=g) + 1j * torch.randn(m, n, dtype=torch.float64, generator=g)
    return a.to(device)


def randr(m, n, seed, device="cuda"):
    g = torch.Generator(device="cpu").manual_seed(seed)
    return torch.randn(m, n, dtype=torch.float64, generator=g).to(device)
