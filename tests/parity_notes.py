"""Notes of the statistical parity tests, printed by conftest.py after the last test."""
NOTES: list[str] = []


def note(line: str) -> None:
    NOTES.append(line)
