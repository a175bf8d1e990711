"""B200-native thermocapillary central-moment phase-field lattice Boltzmann step (arxiv 2401.03041).

The product is the C-ABI CUDA library `libtcp.so` (include/tcp.h, csrc/); this package is its thin
Python binding.  See DESIGN.md.
"""
from .binding import (Simulation, TcpError, make_params, tcp_params, lib, library_path, EXPORTS, tcp_params_default,
                      tcp_workspace_bytes, tcp_create, tcp_create_in, tcp_init_fields,
                      tcp_set_wall_temperature, tcp_set_heat_source, tcp_step, tcp_relax_temperature, tcp_read_fields,
                      tcp_synchronize, tcp_read_pressure_static, TCP_STATIC_SCRATCH_BYTES, tcp_launch_count, tcp_last_step_ms, tcp_pattern_copy_ms, tcp_destroy, tcp_last_error,
                      tcp_set_halo, tcp_halo_phases, tcp_halo_message_bytes, tcp_halo_bytes, tcp_step_begin, tcp_step_advance, tcp_step_end,
                      TCP_OK, TCP_EINVAL, TCP_ENOMEM, TCP_ECUDA, TCP_EUNSUPPORTED, TCP_ESTATE)
