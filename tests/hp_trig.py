"""Table 2 as printed, ``-2 + 2 cos(theta)``, in 60-digit decimal arithmetic: a reference for the
eigenvalues that needs neither the oracle nor the host's long double.  Test infrastructure only."""
from decimal import Decimal, getcontext

getcontext().prec = 60
PI = Decimal("3.14159265358979323846264338327950288419716939937510582097494")


def cos_dec(x: Decimal) -> Decimal:
    """Taylor series of cos; |x| <= 2 pi here, so 60 terms are far more than 60 digits need."""
    term, total, x2 = Decimal(1), Decimal(1), x * x
    for m in range(1, 60):
        term = -term * x2 / ((2 * m - 1) * (2 * m))
        total += term
        if abs(term) < Decimal(10) ** -65:
            break
    return total


def theta(bc: int, k: int, n: int) -> Decimal:
    """Argument of Table 2's cosine: periodic 2 pi k / n, Neumann pi k / n, Dirichlet pi (k + 1) / n."""
    if bc == 0:
        return 2 * PI * k / n
    if bc == 1:
        return PI * k / n
    return PI * (k + 1) / n


def table2_printed(bc: int, k: int, n: int) -> Decimal:
    return -2 + 2 * cos_dec(theta(bc, k, n))
