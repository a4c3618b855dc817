"""Writes rect_pulse_W5_nmax32.txt from the CLOSED FORM of SURVEY.md §8(c) pin P4 (Figure-1 property,
PAPER.md:65, :69).  Imports neither oracle/ nor the CUDA path.

Noiseless rectangular pulse, amplitude A on samples p..p+W-1, zero elsewhere, mu=0, sigma=1, eq. 4:
  t = p-k, 0<=k<Nmax : W+k<=Nmax -> width W+k, SNR A W/sqrt(W+k) ; else width Nmax, SNR A (Nmax-k)/sqrt(Nmax)
  t = p+j, 0<=j<W    : width W-j, SNR A sqrt(W-j)
  elsewhere          : width 1, SNR 0
"""
import math
import os

W, A, NMAX, P, N_T = 5, 3.0, 32, 150, 400


def closed_form(t):
    k = P - t
    if 0 <= k < NMAX:
        if W + k <= NMAX:
            return W + k, A * W / math.sqrt(W + k)
        return NMAX, A * (NMAX - k) / math.sqrt(NMAX)
    j = t - P
    if 0 <= j < W:
        return W - j, A * math.sqrt(W - j)
    return 1, 0.0


if __name__ == "__main__":
    here = os.path.dirname(os.path.abspath(__file__))
    with open(os.path.join(here, "rect_pulse_W5_nmax32.txt"), "w") as f:
        f.write(f"# closed form P4 (PAPER.md:65,:69 Figure-1 property): W={W} A={A} Nmax={NMAX} p={P} n_t={N_T} mu=0 sigma=1 eq.4\n")
        f.write("# t width snr\n")
        for t in range(N_T):
            w, s = closed_form(t)
            f.write(f"{t} {w} {s!r}\n")
