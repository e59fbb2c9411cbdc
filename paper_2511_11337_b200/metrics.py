"""Reporting formulas (PAPER.md "Compression Metrics").  No method arithmetic."""


def compression_ratio(n_orig: int, n_comp: int) -> float:
    """CR = N_orig / N_comp."""
    return n_orig / n_comp


def sigma_ssr(n_orig: float, n_comp: float, seconds: float) -> float:
    """Storage-saving rate = (N_orig - N_comp) / T  (the minus sign is lost in the extracted
    text and is fixed by Table I, see tests/golden/table1.txt).  Units of the inputs per second."""
    return (n_orig - n_comp) / seconds


def bits_per_byte(n_orig: int, n_comp: int) -> float:
    return 8.0 * n_comp / n_orig
