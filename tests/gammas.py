"""The gamma basis of the ABI (SURVEY 8(c) O1 / DESIGN R1), typed here independently of both the
oracle and the CUDA path, as gamma_k = [[0, -i sigma_k], [+i sigma_k, 0]], gamma_t = [[0, 1], [1, 0]]."""
import numpy as np

_s = [np.array([[0, 1], [1, 0]], dtype=complex), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]], dtype=complex)]
_z = np.zeros((2, 2), dtype=complex)
_1 = np.eye(2, dtype=complex)
GAMMA = np.array([np.block([[_z, -1j * s], [1j * s, _z]]) for s in _s] + [np.block([[_z, _1], [_1, _z]])])
GAMMA5 = GAMMA[0] @ GAMMA[1] @ GAMMA[2] @ GAMMA[3]


def sigma(mu, nu):
    return 0.5j * (GAMMA[mu] @ GAMMA[nu] - GAMMA[nu] @ GAMMA[mu])
