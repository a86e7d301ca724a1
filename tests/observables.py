"""Reductions that turn fields into the observables the paper discusses (PAPER.md:473 Stefan interface position, PAPER.md:535
bubbles growing and rising from the heated wall).  Test helpers only: host post-processing, no arithmetic of the method."""
import numpy as np


def interface_x(phi_row):
    """Position (node units, node i at i + 1/2) where phi crosses 1/2 along a row that starts in vapour (phi = 1)."""
    below = np.nonzero(phi_row < 0.5)[0]
    if len(below) == 0 or below[0] == 0:
        return float("nan")
    i = int(below[0])
    a, b = float(phi_row[i - 1]), float(phi_row[i])
    return (i - 1 + 0.5) + (a - 0.5) / (a - b)


def film_thickness(phi):
    """Per column: number of vapour nodes (phi > 1/2) between the heated wall and the first liquid node; wall-normal axis first."""
    liquid = phi <= 0.5
    first = liquid.argmax(axis=0).astype(np.float64)
    first[~liquid.any(axis=0)] = phi.shape[0]
    return first


def detached_bubbles(phi):
    """(count, highest node, nodes) of the connected vapour regions that touch neither the heated wall nor the opposite wall."""
    from scipy import ndimage
    lab, n = ndimage.label(phi > 0.5)
    if n == 0:
        return 0, 0, 0
    attached = set(np.unique(lab[0])) | set(np.unique(lab[-1]))
    free = [k for k in range(1, n + 1) if k not in attached]
    if not free:
        return 0, 0, 0
    mask = np.isin(lab, free)
    top = int(np.nonzero(mask.reshape(mask.shape[0], -1).any(axis=1))[0].max()) + 1
    return len(free), top, int(mask.sum())
